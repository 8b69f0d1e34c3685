"""Thin ctypes binding of the C-ABI library (include/prefixflow.h), same names as the C calls.

Argument marshalling only: every step of the path runs in the CUDA kernels behind the ABI.
PyTorch tensors are used as device-memory handles (data_ptr + strides) and torch streams as
cudaStream_t handles.  There is NO fallback: if libprefixflow.so is missing or a call fails, a
PrefixFlowError is raised.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(_HERE, "libprefixflow.so")

PF_OK, PF_INVALID_ARG, PF_UNSUPPORTED, PF_CUDA_ERROR, PF_WORKSPACE, PF_STATE = range(6)
STATUS_NAMES = {0: "PF_OK", 1: "PF_INVALID_ARG", 2: "PF_UNSUPPORTED", 3: "PF_CUDA_ERROR",
                4: "PF_WORKSPACE", 5: "PF_STATE"}

# every symbol include/prefixflow.h declares
SYMBOLS = ("pf_version", "pf_create", "pf_destroy", "pf_last_error", "pf_set_option",
           "pf_workspace_bytes", "pf_group_begin", "pf_phaseA_fwd", "pf_phaseB_fwd",
           "pf_phaseB_bwd", "pf_phaseC_bwd", "pf_group_end", "pf_offload", "pf_prefetch",
           "pf_counter", "pf_profile_read", "pf_group_mark_cached", "pf_segment_bwd",
           "pf_group_set_prefix_ranges", "pf_rope", "pf_kv_proj_grad", "pf_bwd_split_model",
           "pf_static_scratch_bytes", "pf_causal_bwd_static_max_tokens", "pf_causal_bwd_static")


class PrefixFlowError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


class pf_desc(ctypes.Structure):
    _fields_ = [("n_q_heads", ctypes.c_int32), ("n_kv_heads", ctypes.c_int32),
                ("head_dim", ctypes.c_int32), ("softmax_scale", ctypes.c_float)]


class pf_tensor(ctypes.Structure):
    _fields_ = [("ptr", ctypes.c_void_p), ("stride_tok", ctypes.c_int64),
                ("stride_head", ctypes.c_int64)]


_lib = None


def lib() -> ctypes.CDLL:
    """Load libprefixflow.so (built by `python -m paper_2606_01143_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(SO_PATH):
        raise PrefixFlowError(PF_CUDA_ERROR, f"{SO_PATH} not built; run "
                              "`python -m paper_2606_01143_b200.build` (no fallback path exists)")
    L = ctypes.CDLL(SO_PATH)
    vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
    T = pf_tensor
    pi32 = ctypes.POINTER(ctypes.c_int32)
    L.pf_version.restype = i32
    L.pf_version.argtypes = []
    L.pf_create.restype = i32
    L.pf_create.argtypes = [ctypes.POINTER(vp), i32]
    L.pf_destroy.restype = i32
    L.pf_destroy.argtypes = [vp]
    L.pf_last_error.restype = ctypes.c_char_p
    L.pf_last_error.argtypes = [vp]
    L.pf_set_option.restype = i32
    L.pf_set_option.argtypes = [vp, ctypes.c_char_p, i64]
    L.pf_counter.restype = i64
    L.pf_counter.argtypes = [vp, ctypes.c_char_p]
    L.pf_profile_read.restype = i32
    L.pf_profile_read.argtypes = [vp, i32, ctypes.POINTER(ctypes.c_int64),
                                  ctypes.POINTER(ctypes.c_double)]
    L.pf_workspace_bytes.restype = ctypes.c_size_t
    L.pf_workspace_bytes.argtypes = [ctypes.POINTER(pf_desc), i64, i64]
    L.pf_group_begin.restype = i32
    L.pf_group_begin.argtypes = [vp, ctypes.POINTER(pf_desc), i64, T, T, T, T, vp, ctypes.c_size_t,
                                 vp, ctypes.POINTER(vp)]
    L.pf_phaseA_fwd.restype = i32
    L.pf_phaseA_fwd.argtypes = [vp, T, T, vp, vp]
    L.pf_phaseB_fwd.restype = i32
    L.pf_phaseB_fwd.argtypes = [vp, i32, pi32, T, T, T, T, vp, vp]
    L.pf_phaseB_bwd.restype = i32
    L.pf_phaseB_bwd.argtypes = [vp, i32, pi32, T, T, T, T, vp, T, T, T, T, vp]
    L.pf_phaseC_bwd.restype = i32
    L.pf_phaseC_bwd.argtypes = [vp, T, T, vp, T, T, T, T, vp]
    L.pf_group_end.restype = i32
    L.pf_group_end.argtypes = [vp]
    L.pf_group_mark_cached.restype = i32
    L.pf_group_mark_cached.argtypes = [vp]
    L.pf_group_set_prefix_ranges.restype = i32
    L.pf_group_set_prefix_ranges.argtypes = [vp, i32, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64)]
    L.pf_segment_bwd.restype = i32
    L.pf_segment_bwd.argtypes = [vp, i64, T, T, T, T, vp, T, T, vp, vp, T, T, vp]
    L.pf_bwd_split_model.restype = i32
    L.pf_bwd_split_model.argtypes = [ctypes.POINTER(pf_desc), i64, i32, pi32, i32, pi32, pi32]
    L.pf_rope.restype = i32
    L.pf_rope.argtypes = [vp, i32, pi32, i64, T, i32, i32, ctypes.c_float, i32, vp]
    L.pf_kv_proj_grad.restype = i32
    L.pf_kv_proj_grad.argtypes = [vp, i64, i32, i32, vp, i64, vp, i64, vp, vp]
    L.pf_static_scratch_bytes.restype = ctypes.c_size_t
    L.pf_static_scratch_bytes.argtypes = []
    L.pf_causal_bwd_static_max_tokens.restype = i64
    L.pf_causal_bwd_static_max_tokens.argtypes = [ctypes.POINTER(pf_desc)]
    L.pf_causal_bwd_static.restype = i32
    L.pf_causal_bwd_static.argtypes = [vp, ctypes.POINTER(pf_desc), i64, T, T, T, T, vp, T, T, T, T, vp]
    L.pf_offload.restype = i32
    L.pf_offload.argtypes = [vp, vp, vp, ctypes.c_size_t, vp]
    L.pf_prefetch.restype = i32
    L.pf_prefetch.argtypes = [vp, vp, vp, ctypes.c_size_t, vp]
    _lib = L
    return L


# ---------------------------------------------------------------------------------------------
# marshalling helpers
# ---------------------------------------------------------------------------------------------

def as_tensor(t: Optional[torch.Tensor], dtype=torch.bfloat16) -> pf_tensor:
    """[L, H, d] torch tensor -> pf_tensor (pointer + element strides); None -> NULL."""
    if t is None:
        return pf_tensor(None, 0, 0)
    if t.dim() != 3 or t.dtype != dtype:
        raise PrefixFlowError(PF_INVALID_ARG, f"expected a 3-D {dtype} tensor, got {tuple(t.shape)} {t.dtype}")
    if t.shape[2] > 1 and t.stride(2) != 1:
        raise PrefixFlowError(PF_INVALID_ARG, "last dimension must be contiguous")
    return pf_tensor(t.data_ptr() if t.numel() > 0 else None, t.stride(0), t.stride(1))


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None or t.numel() == 0 else t.data_ptr()


def _stat(t: Optional[torch.Tensor], Hq: int, L: int, name: str):
    """fp32 [Hq, L] statistics tensor (LSE) -> raw pointer.  The C side assumes row stride = L, so a
    column slice of a wider tensor (non-contiguous) must be refused here, not written out of bounds."""
    if L == 0:
        return None
    if (t is None or t.dtype != torch.float32 or tuple(t.shape) != (Hq, L) or not t.is_contiguous()
            or not t.is_cuda):
        raise PrefixFlowError(PF_INVALID_ARG, f"{name} must be a contiguous CUDA float32 tensor of shape "
                              f"({Hq}, {L}), got {None if t is None else (tuple(t.shape), t.dtype, t.is_contiguous())}")
    return t.data_ptr()


def _acc(t: torch.Tensor, like: torch.Tensor, name: str):
    """fp32 accumulator rows [L, Hkv, d], contiguous, same shape as the bf16 tensor `like`."""
    if (t.dtype != torch.float32 or tuple(t.shape) != tuple(like.shape) or not t.is_contiguous()
            or not t.is_cuda):
        raise PrefixFlowError(PF_INVALID_ARG, f"{name} must be a contiguous CUDA float32 tensor of shape "
                              f"{tuple(like.shape)}, got {tuple(t.shape)} {t.dtype}")
    return _ptr(t)


def _flat(t: torch.Tensor, name: str, cuda: bool):
    """Contiguous buffer for a raw byte copy (pf_offload / pf_prefetch)."""
    if not t.is_contiguous() or t.is_cuda != cuda or (not cuda and not t.is_pinned()):
        raise PrefixFlowError(PF_INVALID_ARG, f"{name} must be a contiguous "
                              f"{'CUDA' if cuda else 'pinned host'} tensor")
    return _ptr(t)


def _stream(stream) -> Optional[int]:
    if stream is None:
        stream = torch.cuda.current_stream()
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream or None
    return int(stream) or None


def _cu(cu_seqlens_host: Sequence[int]):
    arr = (ctypes.c_int32 * len(cu_seqlens_host))(*[int(x) for x in cu_seqlens_host])
    return arr


def make_desc(n_q_heads: int, n_kv_heads: int, head_dim: int, softmax_scale: float = 0.0) -> pf_desc:
    return pf_desc(int(n_q_heads), int(n_kv_heads), int(head_dim), float(softmax_scale))


class _Handle:
    """Opaque pf_ctx* / pf_group* plus the owning context (for pf_last_error)."""

    def __init__(self, ptr: int, ctx: Optional["_Handle"] = None):
        self.ptr = ptr
        self.ctx = ctx


def _check(status: int, ctx: Optional[_Handle]):
    if status != PF_OK:
        msg = lib().pf_last_error(ctx.ptr if ctx else None)
        raise PrefixFlowError(status, msg.decode() if msg else "")


# ---------------------------------------------------------------------------------------------
# the C calls, one Python function each
# ---------------------------------------------------------------------------------------------

def pf_version() -> int:
    return int(lib().pf_version())


def pf_create(device: int = 0) -> _Handle:
    out = ctypes.c_void_p()
    st = lib().pf_create(ctypes.byref(out), int(device))
    if st != PF_OK:
        raise PrefixFlowError(st, f"pf_create(device={device}) failed (needs an sm_100 GPU)")
    return _Handle(out.value)


def pf_destroy(ctx: _Handle) -> None:
    _check(lib().pf_destroy(ctx.ptr), None)
    ctx.ptr = None


def pf_last_error(ctx: _Handle) -> str:
    return lib().pf_last_error(ctx.ptr).decode()


def pf_set_option(ctx: _Handle, name: str, value: int) -> None:
    _check(lib().pf_set_option(ctx.ptr, name.encode(), int(value)), ctx)


def pf_counter(ctx: _Handle, name: str) -> int:
    return int(lib().pf_counter(ctx.ptr, name.encode()))


def pf_profile_read(ctx: _Handle, kind: int):
    """(launches, total_ms) of the attention kernels of `kind` (0 fwd, 1 bwd) since the last read."""
    n, ms = ctypes.c_int64(), ctypes.c_double()
    _check(lib().pf_profile_read(ctx.ptr, int(kind), ctypes.byref(n), ctypes.byref(ms)), ctx)
    return int(n.value), float(ms.value)


def pf_workspace_bytes(desc: pf_desc, Lp: int, max_Ls: int) -> int:
    return int(lib().pf_workspace_bytes(ctypes.byref(desc), int(Lp), int(max_Ls)))


def pf_group_begin(ctx: _Handle, desc: pf_desc, Lp: int, K1, V1, gK1, gV1, workspace: torch.Tensor,
                   stream=None) -> _Handle:
    out = ctypes.c_void_p()
    st = lib().pf_group_begin(ctx.ptr, ctypes.byref(desc), int(Lp), as_tensor(K1), as_tensor(V1),
                              as_tensor(gK1, torch.float32), as_tensor(gV1, torch.float32),
                              _ptr(workspace), workspace.numel() * workspace.element_size(),
                              _stream(stream), ctypes.byref(out))
    _check(st, ctx)
    return _Handle(out.value, ctx)


def pf_phaseA_fwd(grp: _Handle, Q1, O1, LSE1, stream=None) -> None:
    _check(lib().pf_phaseA_fwd(grp.ptr, as_tensor(Q1), as_tensor(O1),
                               _stat(LSE1, Q1.shape[1], Q1.shape[0], "LSE1"), _stream(stream)), grp.ctx)


def pf_phaseB_fwd(grp: _Handle, cu_seqlens_host: Sequence[int], Q2, K2, V2, O2, LSE2,
                  stream=None) -> None:
    cu = _cu(cu_seqlens_host)
    _check(lib().pf_phaseB_fwd(grp.ptr, len(cu_seqlens_host) - 1, cu,
                               as_tensor(Q2), as_tensor(K2), as_tensor(V2), as_tensor(O2),
                               _stat(LSE2, Q2.shape[1], Q2.shape[0], "LSE2"), _stream(stream)), grp.ctx)


def pf_phaseB_bwd(grp: _Handle, cu_seqlens_host: Sequence[int], Q2, K2, V2, O2, LSE2, dO2, dQ2, dK2,
                  dV2, stream=None) -> None:
    cu = _cu(cu_seqlens_host)
    _check(lib().pf_phaseB_bwd(grp.ptr, len(cu_seqlens_host) - 1, cu,
                               as_tensor(Q2), as_tensor(K2), as_tensor(V2), as_tensor(O2),
                               _stat(LSE2, Q2.shape[1], Q2.shape[0], "LSE2"), as_tensor(dO2),
                               as_tensor(dQ2), as_tensor(dK2), as_tensor(dV2), _stream(stream)), grp.ctx)


def pf_phaseC_bwd(grp: _Handle, Q1, O1, LSE1, dO1, dQ1, dK1, dV1, stream=None) -> None:
    _check(lib().pf_phaseC_bwd(grp.ptr, as_tensor(Q1), as_tensor(O1),
                               _stat(LSE1, Q1.shape[1], Q1.shape[0], "LSE1"), as_tensor(dO1),
                               as_tensor(dQ1), as_tensor(dK1), as_tensor(dV1), _stream(stream)),
           grp.ctx)


def pf_group_mark_cached(grp: _Handle) -> None:
    _check(lib().pf_group_mark_cached(grp.ptr), grp.ctx)


def pf_group_set_prefix_ranges(grp: _Handle, ranges: Sequence[Sequence[int]]) -> None:
    """ranges: [(start, len), ...] ascending rows of the K1/V1 buffer visible as the prefix."""
    n = len(ranges)
    starts = (ctypes.c_int64 * max(1, n))(*[int(r[0]) for r in ranges])
    lens = (ctypes.c_int64 * max(1, n))(*[int(r[1]) for r in ranges])
    _check(lib().pf_group_set_prefix_ranges(grp.ptr, n, starts, lens), grp.ctx)


def pf_segment_bwd(grp: _Handle, Q, K, V, O, LSE, dO, dQ, accK, accV, dK, dV, stream=None) -> None:
    _check(lib().pf_segment_bwd(grp.ptr, int(Q.shape[0]), as_tensor(Q), as_tensor(K), as_tensor(V),
                                as_tensor(O), _stat(LSE, Q.shape[1], Q.shape[0], "LSE"), as_tensor(dO),
                                as_tensor(dQ), _acc(accK, K, "accK"), _acc(accV, V, "accV"),
                                as_tensor(dK), as_tensor(dV), _stream(stream)), grp.ctx)


def pf_group_end(grp: _Handle) -> None:
    _check(lib().pf_group_end(grp.ptr), grp.ctx)
    grp.ptr = None


def pf_bwd_split_model(desc: pf_desc, Lp: int, cu_seqlens_host: Sequence[int], n_sms: int = 148):
    """(pairs per prefix-tile item, heads per causal-tile item) the backward would use; host-only."""
    a, b = ctypes.c_int32(0), ctypes.c_int32(0)
    st = lib().pf_bwd_split_model(ctypes.byref(desc), int(Lp), len(cu_seqlens_host) - 1, _cu(cu_seqlens_host),
                                  int(n_sms), ctypes.byref(a), ctypes.byref(b))
    if st != PF_OK:
        raise PrefixFlowError(st, "pf_bwd_split_model: invalid arguments")
    return a.value, b.value


def pf_rope(ctx: _Handle, cu_seqlens_host: Sequence[int], pos0: int, X: torch.Tensor, theta_base: float = 10000.0,
            inverse: bool = False, stream=None) -> None:
    """In-place RoPE of a packed bf16 [total, H, d] tensor; row r of sequence s sits at position
    pos0 + (r - cu[s]) (suffix positions continue after the prefix)."""
    _check(lib().pf_rope(ctx.ptr, len(cu_seqlens_host) - 1, _cu(cu_seqlens_host), int(pos0), as_tensor(X), int(X.shape[1]), int(X.shape[2]),
                         float(theta_base), int(bool(inverse)), _stream(stream)), ctx)


def pf_kv_proj_grad(ctx: _Handle, X: torch.Tensor, dY: torch.Tensor, dW: torch.Tensor, stream=None) -> None:
    """dW[d_model, n_cols] (fp32, contiguous) += X[L, d_model]^T dY[L, n_cols]; dY may be a
    [L, Hkv, d] tensor with contiguous (head, d) (one term of dW_K / dW_V)."""
    if dY.dim() == 3:
        if dY.stride(1) != dY.shape[2] or dY.stride(2) != 1:
            raise PrefixFlowError(PF_INVALID_ARG, "pf_kv_proj_grad: dY [L, H, d] must have contiguous (H, d)")
        n_cols, ldy = dY.shape[1] * dY.shape[2], dY.stride(0)
    else:
        n_cols, ldy = dY.shape[1], dY.stride(0)
    if (X.dim() != 2 or X.dtype != torch.bfloat16 or dY.dtype != torch.bfloat16 or X.stride(1) != 1 or
            X.shape[0] != dY.shape[0] or not X.is_cuda or not dY.is_cuda):
        raise PrefixFlowError(PF_INVALID_ARG, "pf_kv_proj_grad: X must be a bf16 CUDA [L, d_model] matrix with as many rows as dY")
    if (dW.dtype != torch.float32 or tuple(dW.shape) != (X.shape[1], n_cols) or not dW.is_contiguous() or not dW.is_cuda):
        raise PrefixFlowError(PF_INVALID_ARG, f"pf_kv_proj_grad: dW must be a contiguous fp32 CUDA [{X.shape[1]}, {n_cols}] matrix")
    _check(lib().pf_kv_proj_grad(ctx.ptr, int(X.shape[0]), int(X.shape[1]), int(n_cols), _ptr(X), int(X.stride(0)),
                                 _ptr(dY), int(ldy), _ptr(dW), _stream(stream)), ctx)


def pf_static_scratch_bytes() -> int:
    return int(lib().pf_static_scratch_bytes())


def pf_causal_bwd_static_max_tokens(desc: pf_desc) -> int:
    return int(lib().pf_causal_bwd_static_max_tokens(ctypes.byref(desc)))


def pf_causal_bwd_static(ctx: _Handle, desc: pf_desc, Q, K, V, O, LSE, dO, dQ, dK, dV, stream=None) -> None:
    """Allocation-free causal backward of one sequence: the workspace is the library's built-in
    32 MiB scratch (include/prefixflow.h); calls that overlap on the GPU race."""
    L = int(Q.shape[0])
    _check(lib().pf_causal_bwd_static(ctx.ptr, ctypes.byref(desc), L, as_tensor(Q), as_tensor(K), as_tensor(V),
                                      as_tensor(O), _stat(LSE, Q.shape[1], L, "LSE"), as_tensor(dO),
                                      as_tensor(dQ), as_tensor(dK), as_tensor(dV), _stream(stream)), ctx)


def pf_offload(ctx: _Handle, src_dev: torch.Tensor, dst_pinned_host: torch.Tensor, stream) -> None:
    nbytes = src_dev.numel() * src_dev.element_size()
    if dst_pinned_host.numel() * dst_pinned_host.element_size() < nbytes:
        raise PrefixFlowError(PF_INVALID_ARG, "pf_offload: destination smaller than source")
    _check(lib().pf_offload(ctx.ptr, _flat(src_dev, "src_dev", True),
                            _flat(dst_pinned_host, "dst_pinned_host", False), nbytes, _stream(stream)), ctx)


def pf_prefetch(ctx: _Handle, src_pinned_host: torch.Tensor, dst_dev: torch.Tensor, stream) -> None:
    nbytes = dst_dev.numel() * dst_dev.element_size()
    if src_pinned_host.numel() * src_pinned_host.element_size() < nbytes:
        raise PrefixFlowError(PF_INVALID_ARG, "pf_prefetch: source smaller than destination")
    _check(lib().pf_prefetch(ctx.ptr, _flat(src_pinned_host, "src_pinned_host", False),
                             _flat(dst_dev, "dst_dev", True), nbytes, _stream(stream)), ctx)
