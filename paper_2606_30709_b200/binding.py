"""ctypes binding of include/hga.h.  Same names as the C entry points; argument marshalling only."""
from __future__ import annotations

import ctypes as C
import dataclasses
import os
from typing import Optional

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_PKG, "libhga.so")
_lib = None

HGA_F32, HGA_BF16 = 0, 1
ROUTE_MEAN, ROUTE_MAX, ROUTE_MAX_FP64 = 0, 1, 2
FLAG_FUSE_Q_ROPE = 1
ATTEND_AUTO, ATTEND_SIMT, ATTEND_TCGEN05, ATTEND_TCGEN05_ITEM, ATTEND_TCGEN05_PAIR = 0, 1, 2, 3, 4


class HgaError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = code
        msg = load_library().hga_status_string(code).decode()
        super().__init__(f"{what}: {msg}")


class _CParams(C.Structure):
    _fields_ = [
        ("batch", C.c_int32), ("seq", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32),
        ("head_dim", C.c_int32), ("chunk", C.c_int32), ("group", C.c_int32), ("n_sink", C.c_int32),
        ("n_local", C.c_int32), ("topk_chunks", C.c_int32), ("topk_groups", C.c_int32), ("n_hi_chunk", C.c_int32),
        ("n_hi_group", C.c_int32), ("io_dtype", C.c_int32), ("out_dtype", C.c_int32), ("attend_impl", C.c_int32),
        ("pos0", C.c_int64), ("rope_base", C.c_double), ("softmax_scale", C.c_float), ("rope_pos_mod", C.c_int32),
        ("route_mode", C.c_int32), ("flags", C.c_int32),
    ]


class _CBuffers(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in (
        "q_raw", "k_raw", "v", "q_rot", "k_rot", "q_pooled", "chunk_sum", "group_sum", "chunk_idx", "chunk_score",
        "n_chunks", "group_idx", "group_score", "n_groups", "out", "lse", "workspace")] + [("workspace_bytes", C.c_size_t)]


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """Load libhga.so (built in-tree by paper_2606_30709_b200/build.py).  Fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise RuntimeError(f"{_LIB_PATH} is missing: build it with `python -m paper_2606_30709_b200.build` "
                           "(or __graft_entry__.build()).  There is no CPU fallback.")
    lib = C.CDLL(_LIB_PATH)
    P, V, I, F = C.POINTER(_CParams), C.c_void_p, C.c_int32, C.c_void_p
    lib.hga_status_string.restype = C.c_char_p
    lib.hga_status_string.argtypes = [C.c_int]
    lib.hga_version.restype = C.c_int32
    lib.hga_default_n_hi.restype = C.c_int32
    lib.hga_default_n_hi.argtypes = [C.c_int32, C.c_double, C.c_int32]
    lib.hga_n_hi_rule.restype = C.c_int32
    lib.hga_n_hi_rule.argtypes = [C.c_int32, C.c_double, C.c_int32, C.c_int32]
    lib.hga_validate.argtypes = [P]
    lib.hga_workspace_bytes.argtypes = [P, C.POINTER(C.c_size_t)]
    lib.hga_rope.argtypes = [P, V, I, V, F, V]
    lib.hga_build_summaries.argtypes = [P, V, V, F, F, V]
    lib.hga_route.argtypes = [P, F, F, F, V, F, V, V, F, V, V, C.c_size_t, V]
    lib.hga_route_static.argtypes = [P, F, F, F, V, F, V, V, F, V, V]
    lib.hga_route_max.argtypes = [P, V, F, F, V, F, V, V, F, V, V, C.c_size_t, V]
    lib.hga_attend.argtypes = [P, V, V, V, V, V, F, V]
    lib.hga_prefill.argtypes = [P, C.POINTER(_CBuffers), V]
    lib.hga_prefill_window.argtypes = [P, C.POINTER(_CBuffers), C.c_int64, C.c_int64, V]
    lib.hga_prefill_profile.argtypes = [P, C.POINTER(_CBuffers), V, C.POINTER(C.c_float)]
    lib.hga_host_plan_create.argtypes = [P, C.POINTER(C.c_void_p)]
    lib.hga_host_prefill.argtypes = [V, V, V, V, V, V, V]
    lib.hga_host_plan_destroy.argtypes = [V]
    lib.hga_host_plan_destroy.restype = None
    lib.hga_host_bytes.argtypes = [P, C.c_int32, C.c_int32, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
    _lib = lib
    return lib


@dataclasses.dataclass
class Params:
    """Mirror of `hga_params` (include/hga.h)."""

    batch: int
    seq: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    chunk: int = 64
    group: int = 16
    n_sink: int = 1
    n_local: int = 1
    topk_chunks: int = 16
    topk_groups: int = 32
    n_hi_chunk: int = -1
    n_hi_group: int = -1
    io_dtype: int = HGA_BF16
    out_dtype: int = HGA_F32
    attend_impl: int = ATTEND_AUTO
    pos0: int = 0
    rope_base: float = 1.0e4
    softmax_scale: float = 0.0
    rope_pos_mod: int = 0
    route_mode: int = 0  # ROUTE_MEAN / ROUTE_MAX / ROUTE_MAX_FP64
    flags: int = 0       # FLAG_FUSE_Q_ROPE: q_rot is not materialised, S4 rotates its query tiles itself (N2)

    def c(self) -> _CParams:
        return _CParams(self.batch, self.seq, self.n_q_heads, self.n_kv_heads, self.head_dim, self.chunk, self.group,
                        self.n_sink, self.n_local, self.topk_chunks, self.topk_groups, self.n_hi_chunk, self.n_hi_group,
                        self.io_dtype, self.out_dtype, self.attend_impl, self.pos0, self.rope_base, self.softmax_scale,
                        self.rope_pos_mod, self.route_mode, self.flags)

    @property
    def n_blocks(self) -> int:
        return self.seq // self.chunk

    @property
    def torch_io(self) -> torch.dtype:
        return torch.bfloat16 if self.io_dtype == HGA_BF16 else torch.float32

    @property
    def torch_out(self) -> torch.dtype:
        return torch.bfloat16 if self.out_dtype == HGA_BF16 else torch.float32

    def replace(self, **kw) -> "Params":
        return dataclasses.replace(self, **kw)


def params_from_workload(w, out_dtype: int = HGA_F32, attend_impl: int = ATTEND_AUTO) -> Params:
    return Params(batch=w.batch, seq=w.seq, n_q_heads=w.n_q_heads, n_kv_heads=w.n_kv_heads, head_dim=w.head_dim,
                  chunk=w.chunk, group=w.group, n_sink=w.n_sink, n_local=w.n_local, topk_chunks=w.topk_chunks,
                  topk_groups=w.topk_groups, io_dtype=HGA_BF16 if w.dtype == "bf16" else HGA_F32, out_dtype=out_dtype,
                  attend_impl=attend_impl, pos0=w.pos0, rope_base=w.rope_base,
                  n_hi_chunk=getattr(w, "n_hi_chunk", -1), n_hi_group=getattr(w, "n_hi_group", -1),
                  rope_pos_mod=getattr(w, "rope_pos_mod", 0), route_mode=int(getattr(w, "route_max", False)))


def _check(code: int, what: str):
    if code != 0:
        raise HgaError(code, what)


def _ptr(t: Optional[torch.Tensor]):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device tensors must be CUDA and contiguous"
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def hga_version() -> int:
    return int(load_library().hga_version())


def hga_default_n_hi(head_dim: int, rope_base: float, span: int) -> int:
    return int(load_library().hga_default_n_hi(head_dim, rope_base, span))


def hga_n_hi_rule(head_dim: int, rope_base: float, span: int, rule: int) -> int:
    return int(load_library().hga_n_hi_rule(head_dim, rope_base, span, rule))


def hga_validate(p: Params) -> int:
    return int(load_library().hga_validate(C.byref(p.c())))


def hga_workspace_bytes(p: Params) -> int:
    n = C.c_size_t(0)
    _check(load_library().hga_workspace_bytes(C.byref(p.c()), C.byref(n)), "hga_workspace_bytes")
    return int(n.value)


def hga_rope(p: Params, x_raw: torch.Tensor, x_rot: Optional[torch.Tensor] = None, pooled=True):
    """S0.  Returns (x_rot, pooled or None).  pooled may be True (allocate), a tensor, or None/False (skip)."""
    assert x_raw.dtype == p.torch_io and x_raw.dim() == 4
    n_heads = x_raw.shape[1]
    if x_rot is None:
        x_rot = torch.empty_like(x_raw)
    if pooled is True:
        pooled = torch.empty((p.batch, p.n_kv_heads, p.n_blocks, p.head_dim), dtype=torch.float32, device=x_raw.device)
    elif pooled is False:
        pooled = None
    _check(load_library().hga_rope(C.byref(p.c()), _ptr(x_raw), n_heads, _ptr(x_rot), _ptr(pooled), _stream()), "hga_rope")
    return x_rot, pooled


def hga_build_summaries(p: Params, k_raw: torch.Tensor, k_rot: Optional[torch.Tensor] = None,
                        chunk_sum: Optional[torch.Tensor] = None, group_sum: Optional[torch.Tensor] = None):
    """S1.  Returns (k_rot, chunk_sum, group_sum)."""
    assert k_raw.dtype == p.torch_io and k_raw.dim() == 4
    dev = k_raw.device
    if k_rot is None:
        k_rot = torch.empty_like(k_raw)
    if chunk_sum is None:
        chunk_sum = torch.empty((p.batch, p.n_kv_heads, p.n_blocks, p.head_dim), dtype=torch.float32, device=dev)
    if group_sum is None:
        group_sum = torch.empty((p.batch, p.n_kv_heads, p.seq // p.group, p.head_dim), dtype=torch.float32, device=dev)
    _check(load_library().hga_build_summaries(C.byref(p.c()), _ptr(k_raw), _ptr(k_rot), _ptr(chunk_sum), _ptr(group_sum),
                                              _stream()), "hga_build_summaries")
    return k_rot, chunk_sum, group_sum


@dataclasses.dataclass
class RouteResult:
    chunk_idx: torch.Tensor
    chunk_score: torch.Tensor
    n_chunks: torch.Tensor
    group_idx: torch.Tensor
    group_score: torch.Tensor
    n_groups: torch.Tensor
    workspace: Optional[torch.Tensor]  # the chunk-score matrix [B, Hkv, n_b, n_b] lives here (lower triangle valid)


ROUTE_STATIC_MAX_BYTES = 16 << 20  # HGA_ROUTE_STATIC_MAX_BYTES


def hga_route_static(p: Params, q_pooled: torch.Tensor, chunk_sum: torch.Tensor, group_sum: torch.Tensor,
                     out: Optional["RouteResult"] = None) -> "RouteResult":
    """S2 + S3 with the library's static device scratch: no workspace argument, no allocation inside the C call.  Pass `out`
    (a RouteResult from an earlier call) to make the Python side allocation-free too."""
    dev = q_pooled.device
    units = (p.batch, p.n_kv_heads, p.n_blocks)
    r = out
    if r is None:
        r = RouteResult(
            chunk_idx=torch.empty(units + (max(p.topk_chunks, 1),), dtype=torch.int32, device=dev),
            chunk_score=torch.empty(units + (max(p.topk_chunks, 1),), dtype=torch.float32, device=dev),
            n_chunks=torch.empty(units, dtype=torch.int32, device=dev),
            group_idx=torch.empty(units + (max(p.topk_groups, 1),), dtype=torch.int32, device=dev),
            group_score=torch.empty(units + (max(p.topk_groups, 1),), dtype=torch.float32, device=dev),
            n_groups=torch.empty(units, dtype=torch.int32, device=dev),
            workspace=None,
        )
    _check(load_library().hga_route_static(C.byref(p.c()), _ptr(q_pooled), _ptr(chunk_sum), _ptr(group_sum),
                                           _ptr(r.chunk_idx), _ptr(r.chunk_score), _ptr(r.n_chunks), _ptr(r.group_idx),
                                           _ptr(r.group_score), _ptr(r.n_groups), _stream()), "hga_route_static")
    return r


def hga_route(p: Params, q_pooled: torch.Tensor, chunk_sum: torch.Tensor, group_sum: torch.Tensor,
              workspace: Optional[torch.Tensor] = None) -> RouteResult:
    """S2 + S3."""
    dev = q_pooled.device
    units = (p.batch, p.n_kv_heads, p.n_blocks)
    ws_bytes = hga_workspace_bytes(p)
    if workspace is None:
        workspace = torch.empty(max(ws_bytes, 16), dtype=torch.uint8, device=dev)
    r = RouteResult(
        chunk_idx=torch.empty(units + (max(p.topk_chunks, 1),), dtype=torch.int32, device=dev),
        chunk_score=torch.empty(units + (max(p.topk_chunks, 1),), dtype=torch.float32, device=dev),
        n_chunks=torch.empty(units, dtype=torch.int32, device=dev),
        group_idx=torch.empty(units + (max(p.topk_groups, 1),), dtype=torch.int32, device=dev),
        group_score=torch.empty(units + (max(p.topk_groups, 1),), dtype=torch.float32, device=dev),
        n_groups=torch.empty(units, dtype=torch.int32, device=dev),
        workspace=workspace,
    )
    _check(load_library().hga_route(C.byref(p.c()), _ptr(q_pooled), _ptr(chunk_sum), _ptr(group_sum), _ptr(r.chunk_idx),
                                    _ptr(r.chunk_score), _ptr(r.n_chunks), _ptr(r.group_idx), _ptr(r.group_score),
                                    _ptr(r.n_groups), _ptr(workspace), workspace.numel(), _stream()), "hga_route")
    return r


def hga_attend(p: Params, q_rot: torch.Tensor, k_rot: torch.Tensor, v: torch.Tensor, group_idx: Optional[torch.Tensor],
               out: Optional[torch.Tensor] = None, lse=True):
    """S4.  Returns (out, lse or None)."""
    assert q_rot.dtype == p.torch_io and k_rot.dtype == p.torch_io and v.dtype == p.torch_io
    if group_idx is not None:
        assert group_idx.dtype == torch.int32
    if out is None:
        out = torch.empty(q_rot.shape, dtype=p.torch_out, device=q_rot.device)
    if lse is True:
        lse = torch.empty(q_rot.shape[:3], dtype=torch.float32, device=q_rot.device)
    elif lse is False:
        lse = None
    _check(load_library().hga_attend(C.byref(p.c()), _ptr(q_rot), _ptr(k_rot), _ptr(v), _ptr(group_idx), _ptr(out),
                                     _ptr(lse), _stream()), "hga_attend")
    return out, lse


@dataclasses.dataclass
class PrefillBuffers:
    """Device buffers of one prefill pass (mirror of `hga_buffers`)."""

    q_rot: Optional[torch.Tensor]
    k_rot: torch.Tensor
    q_pooled: torch.Tensor
    chunk_sum: torch.Tensor
    group_sum: torch.Tensor
    chunk_idx: torch.Tensor
    chunk_score: torch.Tensor
    n_chunks: torch.Tensor
    group_idx: torch.Tensor
    group_score: torch.Tensor
    n_groups: torch.Tensor
    out: torch.Tensor
    lse: torch.Tensor
    workspace: torch.Tensor

    @staticmethod
    def allocate(p: Params, device="cuda") -> "PrefillBuffers":
        units = (p.batch, p.n_kv_heads, p.n_blocks)
        f32, i32 = torch.float32, torch.int32
        e = lambda shape, dt: torch.empty(shape, dtype=dt, device=device)
        return PrefillBuffers(
            # with FLAG_FUSE_Q_ROPE the rotated queries are never written: no buffer (a NULL pointer at the C boundary)
            q_rot=None if p.flags & FLAG_FUSE_Q_ROPE else e((p.batch, p.n_q_heads, p.seq, p.head_dim), p.torch_io),
            k_rot=e((p.batch, p.n_kv_heads, p.seq, p.head_dim), p.torch_io),
            q_pooled=e(units + (p.head_dim,), f32), chunk_sum=e(units + (p.head_dim,), f32),
            group_sum=e((p.batch, p.n_kv_heads, p.seq // p.group, p.head_dim), f32),
            chunk_idx=e(units + (max(p.topk_chunks, 1),), i32), chunk_score=e(units + (max(p.topk_chunks, 1),), f32),
            n_chunks=e(units, i32),
            group_idx=e(units + (max(p.topk_groups, 1),), i32), group_score=e(units + (max(p.topk_groups, 1),), f32),
            n_groups=e(units, i32),
            out=e((p.batch, p.n_q_heads, p.seq, p.head_dim), p.torch_out),
            lse=e((p.batch, p.n_q_heads, p.seq), f32),
            workspace=torch.empty(max(hga_workspace_bytes(p), 16), dtype=torch.uint8, device=device),
        )


def _cbuffers(q_raw, k_raw, v, buf, want_lse):
    cb = _CBuffers()
    cb.q_raw, cb.k_raw, cb.v = q_raw.data_ptr(), k_raw.data_ptr(), v.data_ptr()
    for name in ("q_rot", "k_rot", "q_pooled", "chunk_sum", "group_sum", "chunk_idx", "chunk_score", "n_chunks",
                 "group_idx", "group_score", "n_groups", "out", "workspace"):
        t = getattr(buf, name)
        setattr(cb, name, t.data_ptr() if t is not None else None)
    cb.lse = buf.lse.data_ptr() if want_lse else None
    cb.workspace_bytes = buf.workspace.numel()
    return cb


def hga_prefill(p: Params, q_raw: torch.Tensor, k_raw: torch.Tensor, v: torch.Tensor,
                buf: Optional[PrefillBuffers] = None, want_lse: bool = True) -> PrefillBuffers:
    """S0..S4 on the current stream (one C call)."""
    assert q_raw.dtype == p.torch_io and k_raw.dtype == p.torch_io and v.dtype == p.torch_io
    if buf is None:
        buf = PrefillBuffers.allocate(p, q_raw.device)
    cb = _cbuffers(q_raw, k_raw, v, buf, want_lse)
    _check(load_library().hga_prefill(C.byref(p.c()), C.byref(cb), _stream()), "hga_prefill")
    return buf


def hga_prefill_window(p: Params, q_raw: torch.Tensor, k_raw: torch.Tensor, v: torch.Tensor, buf: PrefillBuffers,
                       t_begin: int, t_end: int, want_lse: bool = True) -> PrefillBuffers:
    """One streaming step over tokens [t_begin, t_end) of the cache held in (q_raw, k_raw, v, buf) (one C call)."""
    assert q_raw.dtype == p.torch_io and k_raw.dtype == p.torch_io and v.dtype == p.torch_io
    cb = _cbuffers(q_raw, k_raw, v, buf, want_lse)
    _check(load_library().hga_prefill_window(C.byref(p.c()), C.byref(cb), t_begin, t_end, _stream()),
           "hga_prefill_window")
    return buf


def hga_prefill_profile(p: Params, q_raw: torch.Tensor, k_raw: torch.Tensor, v: torch.Tensor, buf: PrefillBuffers,
                        want_lse: bool = True):
    """hga_prefill with events between its launches; synchronises and returns [S0+S1, S2+S3, S4] in ms."""
    cb = _cbuffers(q_raw, k_raw, v, buf, want_lse)
    ms = (C.c_float * 3)()
    _check(load_library().hga_prefill_profile(C.byref(p.c()), C.byref(cb), _stream(), ms), "hga_prefill_profile")
    return [float(x) for x in ms]


class HostPlan:
    """Host-buffer path (hga_host_plan_*): H2D copies, S0..S4, D2H copies inside one C call."""

    def __init__(self, p: Params):
        self.p = p
        self._h = C.c_void_p(None)
        _check(load_library().hga_host_plan_create(C.byref(p.c()), C.byref(self._h)), "hga_host_plan_create")
        h2d, d2h = C.c_size_t(0), C.c_size_t(0)
        _check(load_library().hga_host_bytes(C.byref(p.c()), 0, 0, C.byref(h2d), C.byref(d2h)), "hga_host_bytes")
        self.h2d_bytes, self.d2h_bytes = int(h2d.value), int(d2h.value)

    def prefill(self, q_host: torch.Tensor, k_host: torch.Tensor, v_host: torch.Tensor, out_host: torch.Tensor,
                group_idx_host: Optional[torch.Tensor] = None, lse_host: Optional[torch.Tensor] = None):
        for t in (q_host, k_host, v_host, out_host):
            assert not t.is_cuda and t.is_contiguous()
        hp = lambda t: None if t is None else C.c_void_p(t.data_ptr())
        _check(load_library().hga_host_prefill(self._h, hp(q_host), hp(k_host), hp(v_host), hp(out_host),
                                               hp(group_idx_host), hp(lse_host)), "hga_host_prefill")
        return out_host

    def close(self):
        if self._h:
            load_library().hga_host_plan_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
