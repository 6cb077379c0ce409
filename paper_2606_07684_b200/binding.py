"""ctypes binding of libscd.so (include/scd.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; this module turns
torch tensors into device pointers and Python lists into the C structs, nothing else.
PyTorch is used for device memory and streams.  If libscd.so is missing the import
fails loudly -- there is no CPU or eager fallback.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence, Tuple

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libscd.so")

# enums (include/scd.h)
SCD_OK = 0
SCD_F32, SCD_BF16, SCD_E4M3_ROWSCALE = 0, 1, 2
SCD_REUSE, SCD_PATCH = 0, 1
SCD_BRANCH_K, SCD_BRANCH_V, SCD_BRANCH_H = 0, 1, 2
SCD_ROPE_HALF, SCD_ROPE_INTERLEAVED = 0, 1
SCD_ACT_IDENTITY, SCD_ACT_SILU = 0, 1
SCD_NORM_NONE, SCD_NORM_RMS = 0, 1
SCD_MAX_LAYERS = 128
STATUS_NAMES = {0: "SCD_OK", 1: "SCD_E_ARG", 2: "SCD_E_SHAPE", 3: "SCD_E_UNSUPPORTED", 4: "SCD_E_ALIGN",
                5: "SCD_E_WORKSPACE", 6: "SCD_E_CUDA", 7: "SCD_E_NOMEM"}
NO_SCALE = C.c_size_t(-1).value

# every symbol include/scd.h declares
EXPORTS = ["scd_plan", "scd_plan_destroy", "scd_plan_query", "scd_plan_code_segment", "scd_code_layout",
           "scd_encode", "scd_reuse_decode", "scd_patch", "scd_encode_layers", "scd_reuse_decode_layers",
           "scd_patch_layers", "scd_patch_static", "scd_last_launch_count", "scd_profile_enable",
           "scd_profile_fetch", "scd_last_error", "scd_version",
           "scd_int4_layout", "scd_int4_quantize", "scd_int4_dequantize_paged",
           "scd_fit_query", "scd_fit_reuse", "scd_struct_size"]


class ModelDesc(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("d_model", C.c_int32), ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("block_size", C.c_int32), ("max_position", C.c_int32), ("state_dtype", C.c_int32),
                ("code_dtype", C.c_int32), ("rope_theta_producer", C.c_double), ("rope_theta_consumer", C.c_double),
                ("rope_style", C.c_int32), ("k_is_roped", C.c_int32), ("rope_on_reuse_k", C.c_int32),
                ("patch_act", C.c_int32), ("patch_norm", C.c_int32), ("rms_eps", C.c_float),
                ("reuse_per_head", C.c_int32)]


class LayerDesc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("r_k", C.c_int32), ("r_v", C.c_int32),
                ("enc_k", C.c_void_p), ("enc_v", C.c_void_p), ("dec_k", C.c_void_p), ("dec_v", C.c_void_p),
                ("mean_src_k", C.c_void_p), ("mean_src_v", C.c_void_p),
                ("mean_dst_k", C.c_void_p), ("mean_dst_v", C.c_void_p),
                ("r_h", C.c_int32), ("d_aligner", C.c_int32),
                ("enc_h", C.c_void_p), ("mean_src_h", C.c_void_p),
                ("w1", C.c_void_p), ("b1", C.c_void_p), ("w2", C.c_void_p), ("b2", C.c_void_p),
                ("norm_gamma", C.c_void_p), ("w_k", C.c_void_p), ("w_v", C.c_void_p),
                ("b_k", C.c_void_p), ("b_v", C.c_void_p)]


class BatchDesc(C.Structure):
    _fields_ = [("n_seqs", C.c_int32), ("total_tokens", C.c_int32), ("max_seqlen", C.c_int32),
                ("max_pages_per_seq", C.c_int32), ("cu_seqlens", C.c_void_p), ("page_table", C.c_void_p),
                ("pos_offset", C.c_void_p), ("max_pos_offset", C.c_int32)]


class SrcDesc(C.Structure):
    _fields_ = [("k", C.POINTER(C.c_void_p)), ("v", C.POINTER(C.c_void_p)), ("h", C.POINTER(C.c_void_p)),
                ("kv_token_stride", C.c_int64), ("kv_head_stride", C.c_int64), ("h_token_stride", C.c_int64),
                ("page_table", C.c_void_p), ("max_pages_per_seq", C.c_int32), ("n_blocks", C.c_int32)]


class PagedKV(C.Structure):
    _fields_ = [("k_pool", C.POINTER(C.c_void_p)), ("v_pool", C.POINTER(C.c_void_p)), ("n_blocks", C.c_int32),
                ("pool_e4m3", C.c_int32), ("k_scale", C.POINTER(C.c_void_p)), ("v_scale", C.POINTER(C.c_void_p))]


class Int4Desc(C.Structure):
    _fields_ = [("n_kv_heads", C.c_int32), ("head_dim", C.c_int32), ("block_size", C.c_int32), ("group", C.c_int32)]


class FitDesc(C.Structure):
    _fields_ = [("width", C.c_int32), ("rank", C.c_int32), ("center", C.c_int32), ("lam_rel", C.c_float),
                ("state_dtype", C.c_int32), ("out_dtype", C.c_int32)]


class ScdError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2606_07684_b200.build` "
                          "(the codec has no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, sz = C.c_void_p, C.c_int32, C.c_size_t
    psz, pi32 = C.POINTER(C.c_size_t), C.POINTER(C.c_int32)
    lib.scd_plan.argtypes = [C.POINTER(ModelDesc), C.POINTER(LayerDesc), vp, C.POINTER(vp)]
    lib.scd_plan_destroy.argtypes = [vp]
    lib.scd_plan_query.argtypes = [vp, i32, psz, psz, psz]
    lib.scd_plan_code_segment.argtypes = [vp, i32, i32, i32, psz, psz, pi32]
    lib.scd_code_layout.argtypes = [C.POINTER(ModelDesc), C.POINTER(LayerDesc), i32, i32, i32, psz, psz, pi32, psz, psz]
    lib.scd_encode.argtypes = [vp, C.POINTER(BatchDesc), C.POINTER(SrcDesc), vp, vp]
    lib.scd_reuse_decode.argtypes = [vp, C.POINTER(BatchDesc), vp, C.POINTER(PagedKV), vp]
    lib.scd_patch.argtypes = [vp, C.POINTER(BatchDesc), vp, C.POINTER(PagedKV), vp, sz, vp]
    lib.scd_encode_layers.argtypes = [vp, C.POINTER(BatchDesc), C.POINTER(SrcDesc), vp, i32, i32, vp]
    lib.scd_reuse_decode_layers.argtypes = [vp, C.POINTER(BatchDesc), vp, C.POINTER(PagedKV), i32, i32, vp]
    lib.scd_patch_layers.argtypes = [vp, C.POINTER(BatchDesc), vp, C.POINTER(PagedKV), vp, sz, i32, i32, vp]
    lib.scd_patch_static.argtypes = [vp, C.POINTER(BatchDesc), vp, C.POINTER(PagedKV), vp]
    lib.scd_patch_static.restype = C.c_int
    for name in ("scd_plan", "scd_plan_destroy", "scd_plan_query", "scd_plan_code_segment", "scd_code_layout",
                 "scd_encode", "scd_reuse_decode", "scd_patch"):
        getattr(lib, name).restype = C.c_int
    lib.scd_int4_layout.argtypes = [C.POINTER(Int4Desc), i32, i32, psz, psz, psz, psz]
    lib.scd_int4_quantize.argtypes = [C.POINTER(Int4Desc), i32, i32, C.POINTER(vp), C.c_int64, vp, vp]
    lib.scd_int4_dequantize_paged.argtypes = [C.POINTER(Int4Desc), C.POINTER(BatchDesc), i32, vp, C.POINTER(vp), i32, vp]
    for name in ("scd_int4_layout", "scd_int4_quantize", "scd_int4_dequantize_paged"):
        getattr(lib, name).restype = C.c_int
    lib.scd_fit_query.argtypes = [C.POINTER(FitDesc), C.c_int64, psz]
    lib.scd_fit_reuse.argtypes = [C.POINTER(FitDesc), vp, vp, C.c_int64, C.c_int64, vp, vp, vp, vp, vp, vp, vp, sz, pi32, vp]
    lib.scd_fit_query.restype = C.c_int
    lib.scd_fit_reuse.restype = C.c_int
    lib.scd_last_launch_count.restype = C.c_int32
    lib.scd_profile_enable.argtypes = [i32]
    lib.scd_profile_enable.restype = C.c_int
    lib.scd_profile_fetch.argtypes = [C.POINTER(C.c_float), pi32, i32]
    lib.scd_profile_fetch.restype = C.c_int32
    lib.scd_struct_size.argtypes = [i32]
    lib.scd_struct_size.restype = C.c_int32
    for which, cls in enumerate((ModelDesc, LayerDesc, BatchDesc, SrcDesc, PagedKV, Int4Desc, FitDesc)):
        if lib.scd_struct_size(which) != C.sizeof(cls):
            raise ImportError(f"libscd.so and binding.py disagree on the layout of {cls.__name__}: "
                              f"{lib.scd_struct_size(which)} vs {C.sizeof(cls)} bytes (rebuild the library)")
    lib.scd_last_error.restype = C.c_char_p
    lib.scd_version.restype = C.c_char_p
    return lib


lib = _load()


def _check(st: int) -> None:
    if st != SCD_OK:
        raise ScdError(st, lib.scd_last_error().decode())


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream or None


def model_desc(*, n_layers, d_model, n_kv_heads, head_dim, max_position, state_dtype, code_dtype,
               rope_theta_producer, rope_theta_consumer=None, block_size=16, rope_style=SCD_ROPE_HALF,
               k_is_roped=1, rope_on_reuse_k=1, patch_act=SCD_ACT_SILU, patch_norm=SCD_NORM_RMS,
               rms_eps=1e-5, reuse_per_head=0) -> ModelDesc:
    return ModelDesc(n_layers, d_model, n_kv_heads, head_dim, block_size, max_position, state_dtype, code_dtype,
                     float(rope_theta_producer),
                     float(rope_theta_producer if rope_theta_consumer is None else rope_theta_consumer),
                     rope_style, int(k_is_roped), int(rope_on_reuse_k), patch_act, patch_norm, float(rms_eps),
                     int(reuse_per_head))


def reuse_layer_desc(*, enc_k, enc_v, dec_k, dec_v, mean_src_k=None, mean_src_v=None, mean_dst_k=None,
                     mean_dst_v=None) -> LayerDesc:
    d = LayerDesc()
    d.kind, d.r_k, d.r_v = SCD_REUSE, enc_k.shape[1], enc_v.shape[1]
    d.enc_k, d.enc_v, d.dec_k, d.dec_v = _ptr(enc_k), _ptr(enc_v), _ptr(dec_k), _ptr(dec_v)
    d.mean_src_k, d.mean_src_v = _ptr(mean_src_k), _ptr(mean_src_v)
    d.mean_dst_k, d.mean_dst_v = _ptr(mean_dst_k), _ptr(mean_dst_v)
    d._keep = (enc_k, enc_v, dec_k, dec_v, mean_src_k, mean_src_v, mean_dst_k, mean_dst_v)
    return d


def patch_layer_desc(*, enc_h, w1, w2, w_k, w_v, mean_src_h=None, b1=None, b2=None, norm_gamma=None, b_k=None,
                     b_v=None) -> LayerDesc:
    d = LayerDesc()
    d.kind, d.r_h, d.d_aligner = SCD_PATCH, enc_h.shape[1], w1.shape[1]
    d.enc_h, d.mean_src_h = _ptr(enc_h), _ptr(mean_src_h)
    d.w1, d.b1, d.w2, d.b2 = _ptr(w1), _ptr(b1), _ptr(w2), _ptr(b2)
    d.norm_gamma, d.w_k, d.w_v, d.b_k, d.b_v = _ptr(norm_gamma), _ptr(w_k), _ptr(w_v), _ptr(b_k), _ptr(b_v)
    d._keep = (enc_h, mean_src_h, w1, b1, w2, b2, norm_gamma, w_k, w_v, b_k, b_v)
    return d


def batch_desc(cu_seqlens: torch.Tensor, page_table: Optional[torch.Tensor], pos_offset: Optional[torch.Tensor],
               seqlens: Sequence[int], max_pos_offset: int = 0) -> BatchDesc:
    b = BatchDesc()
    b.n_seqs = len(seqlens)
    b.total_tokens = int(sum(seqlens))
    b.max_seqlen = max(seqlens) if len(seqlens) else 0
    b.max_pages_per_seq = 0 if page_table is None else page_table.shape[1]
    b.cu_seqlens, b.page_table, b.pos_offset = _ptr(cu_seqlens), _ptr(page_table), _ptr(pos_offset)
    b.max_pos_offset = int(max_pos_offset)
    b._keep = (cu_seqlens, page_table, pos_offset)
    return b


def _ptr_array(tensors: Sequence[Optional[torch.Tensor]]):
    arr = (C.c_void_p * len(tensors))()
    for i, t in enumerate(tensors):
        arr[i] = _ptr(t)
    return arr


def scd_code_layout(model: ModelDesc, layers: Sequence[LayerDesc], total_tokens: int, layer: int = -1,
                    branch: int = 0):
    """(offset, scale_offset, rank, code_bytes, payload_bytes); pure host arithmetic."""
    arr = (LayerDesc * len(layers))(*layers)
    off, soff, cb, pb = C.c_size_t(0), C.c_size_t(0), C.c_size_t(0), C.c_size_t(0)
    rank = C.c_int32(0)
    _check(lib.scd_code_layout(C.byref(model), arr, total_tokens, layer, branch, C.byref(off), C.byref(soff),
                               C.byref(rank), C.byref(cb), C.byref(pb)))
    return off.value, soff.value, rank.value, cb.value, pb.value


class Plan:
    """Owner of an scd_plan_t* (scd_plan / scd_plan_destroy)."""

    def __init__(self, model: ModelDesc, layers: Sequence[LayerDesc], stream=None):
        self.model = model
        self.n_layers = model.n_layers
        arr = (LayerDesc * len(layers))(*layers)
        h = C.c_void_p()
        _check(lib.scd_plan(C.byref(model), arr, _stream_ptr(stream), C.byref(h)))
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            lib.scd_plan_destroy(self.handle)
            self.handle = None

    __del__ = close

    def query(self, total_tokens: int) -> Tuple[int, int, int]:
        cb, ws, pb = C.c_size_t(0), C.c_size_t(0), C.c_size_t(0)
        _check(lib.scd_plan_query(self.handle, total_tokens, C.byref(cb), C.byref(ws), C.byref(pb)))
        return cb.value, ws.value, pb.value

    def code_segment(self, layer: int, branch: int, total_tokens: int) -> Tuple[int, int, int]:
        off, soff, rank = C.c_size_t(0), C.c_size_t(0), C.c_int32(0)
        _check(lib.scd_plan_code_segment(self.handle, layer, branch, total_tokens, C.byref(off), C.byref(soff),
                                         C.byref(rank)))
        return off.value, soff.value, rank.value


def scd_plan(model: ModelDesc, layers: Sequence[LayerDesc], stream=None) -> Plan:
    return Plan(model, layers, stream)


def scd_encode(plan: Plan, batch: BatchDesc, k: Sequence[Optional[torch.Tensor]],
               v: Sequence[Optional[torch.Tensor]], h: Sequence[Optional[torch.Tensor]], codes: torch.Tensor,
               kv_token_stride: int, kv_head_stride: int, h_token_stride: int, stream=None, layers=None,
               src_page_table: Optional[torch.Tensor] = None, src_n_blocks: int = 0) -> int:
    """`layers` = (begin, end): the layer-streamed variant scd_encode_layers.  `src_page_table` [n_seqs, max_pages]
    int32: k / v are the producer's paged pools and rows are gathered through it."""
    src = SrcDesc(_ptr_array(k), _ptr_array(v), _ptr_array(h), kv_token_stride, kv_head_stride, h_token_stride,
                  _ptr(src_page_table), 0 if src_page_table is None else src_page_table.shape[1], src_n_blocks)
    if layers is None:
        _check(lib.scd_encode(plan.handle, C.byref(batch), C.byref(src), _ptr(codes), _stream_ptr(stream)))
    else:
        _check(lib.scd_encode_layers(plan.handle, C.byref(batch), C.byref(src), _ptr(codes), layers[0], layers[1],
                                     _stream_ptr(stream)))
    return lib.scd_last_launch_count()


def _paged_kv(k_pool, v_pool, n_blocks, k_scale, v_scale) -> PagedKV:
    if k_scale is None:
        return PagedKV(_ptr_array(k_pool), _ptr_array(v_pool), n_blocks, 0, None, None)
    return PagedKV(_ptr_array(k_pool), _ptr_array(v_pool), n_blocks, 1, _ptr_array(k_scale), _ptr_array(v_scale))


def scd_reuse_decode(plan: Plan, batch: BatchDesc, codes: torch.Tensor, k_pool: Sequence[Optional[torch.Tensor]],
                     v_pool: Sequence[Optional[torch.Tensor]], n_blocks: int, stream=None, layers=None,
                     k_scale=None, v_scale=None) -> int:
    """k_scale / v_scale (lists of fp32 tensors [n_blocks, bs, H_kv]): the pools are e4m3 bytes (fp8 pools)."""
    kv = _paged_kv(k_pool, v_pool, n_blocks, k_scale, v_scale)
    if layers is None:
        _check(lib.scd_reuse_decode(plan.handle, C.byref(batch), _ptr(codes), C.byref(kv), _stream_ptr(stream)))
    else:
        _check(lib.scd_reuse_decode_layers(plan.handle, C.byref(batch), _ptr(codes), C.byref(kv), layers[0], layers[1],
                                           _stream_ptr(stream)))
    return lib.scd_last_launch_count()


PATCH_STATIC_WORKSPACE_BYTES = 32 << 20        # SCD_PATCH_STATIC_WORKSPACE_BYTES (include/scd.h)


def scd_patch_static(plan: Plan, batch: BatchDesc, codes: torch.Tensor, k_pool: Sequence[Optional[torch.Tensor]],
                     v_pool: Sequence[Optional[torch.Tensor]], n_blocks: int, stream=None, k_scale=None, v_scale=None) -> int:
    """scd_patch with its intermediates in the library's static device array: no workspace argument, no allocation;
    calls that overlap on the GPU race on that array (include/scd.h)."""
    kv = _paged_kv(k_pool, v_pool, n_blocks, k_scale, v_scale)
    _check(lib.scd_patch_static(plan.handle, C.byref(batch), _ptr(codes), C.byref(kv), _stream_ptr(stream)))
    return lib.scd_last_launch_count()


def scd_patch(plan: Plan, batch: BatchDesc, codes: torch.Tensor, k_pool: Sequence[Optional[torch.Tensor]],
              v_pool: Sequence[Optional[torch.Tensor]], n_blocks: int, workspace: Optional[torch.Tensor],
              stream=None, layers=None, k_scale=None, v_scale=None) -> int:
    kv = _paged_kv(k_pool, v_pool, n_blocks, k_scale, v_scale)
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    if layers is None:
        _check(lib.scd_patch(plan.handle, C.byref(batch), _ptr(codes), C.byref(kv), _ptr(workspace), ws_bytes,
                             _stream_ptr(stream)))
    else:
        _check(lib.scd_patch_layers(plan.handle, C.byref(batch), _ptr(codes), C.byref(kv), _ptr(workspace), ws_bytes,
                                    layers[0], layers[1], _stream_ptr(stream)))
    return lib.scd_last_launch_count()


def scd_int4_layout(desc: Int4Desc, total_tokens: int, n_tensors: int):
    """(tensor_stride, meta_offset, total_bytes, payload_bytes); pure host arithmetic."""
    v = [C.c_size_t(0) for _ in range(4)]
    _check(lib.scd_int4_layout(C.byref(desc), total_tokens, n_tensors, *[C.byref(x) for x in v]))
    return tuple(x.value for x in v)


def scd_int4_quantize(desc: Int4Desc, total_tokens: int, src: Sequence[torch.Tensor], token_stride: int,
                      packed: torch.Tensor, stream=None) -> int:
    _check(lib.scd_int4_quantize(C.byref(desc), total_tokens, len(src), _ptr_array(src), token_stride, _ptr(packed),
                                 _stream_ptr(stream)))
    return lib.scd_last_launch_count()


def scd_int4_dequantize_paged(desc: Int4Desc, batch: BatchDesc, packed: torch.Tensor, pools: Sequence[torch.Tensor],
                              n_blocks: int, stream=None) -> int:
    _check(lib.scd_int4_dequantize_paged(C.byref(desc), C.byref(batch), len(pools), _ptr(packed), _ptr_array(pools),
                                         n_blocks, _stream_ptr(stream)))
    return lib.scd_last_launch_count()


def scd_fit_query(desc: FitDesc, n_rows: int) -> int:
    ws = C.c_size_t(0)
    _check(lib.scd_fit_query(C.byref(desc), n_rows, C.byref(ws)))
    return ws.value


def scd_fit_reuse(desc: FitDesc, a: torch.Tensor, b: torch.Tensor, n_rows: int, row_stride: int, w_enc: torch.Tensor,
                  w_dec_a: Optional[torch.Tensor], w_dec_b: torch.Tensor, mu_a: Optional[torch.Tensor],
                  mu_b: Optional[torch.Tensor], sigma: Optional[torch.Tensor], workspace: torch.Tensor, stream=None) -> int:
    """Returns the Jacobi sweeps (joint solve, ridge solve).  Synchronises the stream (not a hot call)."""
    sweeps = (C.c_int32 * 2)()
    _check(lib.scd_fit_reuse(C.byref(desc), _ptr(a), _ptr(b), n_rows, row_stride, _ptr(w_enc), _ptr(w_dec_a), _ptr(w_dec_b),
                             _ptr(mu_a), _ptr(mu_b), _ptr(sigma), _ptr(workspace),
                             workspace.numel() * workspace.element_size(), sweeps, _stream_ptr(stream)))
    return sweeps[0], sweeps[1]


def profile_enable(on: bool) -> None:
    _check(lib.scd_profile_enable(int(on)))


def profile_fetch(max_launches: int = 4096):
    """[(kernel_id, ms)] for every launch since the last fetch (synchronises their events)."""
    ms = (C.c_float * max_launches)()
    ids = (C.c_int32 * max_launches)()
    n = min(lib.scd_profile_fetch(ms, ids, max_launches), max_launches)
    return [(ids[i], ms[i]) for i in range(n)]


def version() -> str:
    return lib.scd_version().decode()
