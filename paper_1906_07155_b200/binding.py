"""Thin ctypes binding of libraf.so (include/raf.h).  Argument marshalling only: every step of the
path (level assignment, bucketing, forward gather, backward scatter, zero-fill) runs in the CUDA
kernels behind the C ABI.  PyTorch is used for device memory and the current stream, nothing else.

There is NO fallback: if libraf.so is missing or a call returns a negative status, this raises.
Function names equal the C entry points.
"""
import ctypes
import os
from typing import List, Optional, Sequence, Tuple

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libraf.so")

RAF_F32, RAF_F16, RAF_BF16 = 0, 1, 2
RAF_ACCUMULATE, RAF_DETERMINISTIC, RAF_ATOMIC, RAF_REUSE_PREP, RAF_NO_PREP = 1, 2, 4, 8, 16
RAF_PULL_STRIP, RAF_PULL_TILE, RAF_REPACK = 32, 64, 128
RAF_SOFT_LINEAR, RAF_SOFT_GAUSSIAN = 1, 2
_DTYPES = {torch.float32: RAF_F32, torch.float16: RAF_F16, torch.bfloat16: RAF_BF16}

EXPORTS = [
    "roi_align_fpn_workspace_bytes", "roi_fpn_assign_levels", "roi_align_fpn_forward",
    "roi_align_fpn_forward_ex", "roi_align_fpn_backward", "roi_align_fpn_backward_ex", "roi_align_fpn_host_arena_bytes", "roi_align_fpn_forward_host",
    "roi_align_fpn_backward_host", "roi_align_fpn_strerror", "roi_align_fpn_launch_count",
    "roi_pool_fpn_forward", "roi_pool_fpn_backward", "roi_nms_workspace_bytes", "roi_nms", "roi_soft_nms",
    "roi_align_fpn_repack_bytes", "roi_deform_pool_fpn_forward", "roi_deform_pool_fpn_backward",
    "roi_align_fc_fpn_forward", "roi_align_fpn_backward_static",
]


class RafLevel(ctypes.Structure):
    _fields_ = [("data", ctypes.c_void_p), ("n", ctypes.c_int32), ("c", ctypes.c_int32),
                ("h", ctypes.c_int32), ("w", ctypes.c_int32), ("sn", ctypes.c_int64),
                ("sc", ctypes.c_int64), ("sh", ctypes.c_int64), ("sw", ctypes.c_int64),
                ("spatial_scale", ctypes.c_float)]


class RafError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: raf_status {status} ({strerror(status)})")


_lib = None


def lib() -> ctypes.CDLL:
    """Load libraf.so; fails loudly if the CUDA library has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not found: build it with "
                               "`python -m paper_1906_07155_b200.build` (no CPU fallback exists)")
        L = ctypes.CDLL(LIB_PATH)
        L.roi_align_fpn_workspace_bytes.restype = ctypes.c_size_t
        L.roi_align_fpn_workspace_bytes.argtypes = [ctypes.c_int] * 6
        L.roi_align_fpn_repack_bytes.restype = ctypes.c_size_t
        L.roi_align_fpn_repack_bytes.argtypes = [ctypes.c_void_p] + [ctypes.c_int] * 5
        L.roi_align_fpn_host_arena_bytes.restype = ctypes.c_size_t
        L.roi_align_fpn_host_arena_bytes.argtypes = [ctypes.c_void_p] + [ctypes.c_int] * 7
        L.roi_fpn_assign_levels.restype = ctypes.c_int
        L.roi_fpn_assign_levels.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_float,
                                            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                            ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p]
        fwd_args = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_int,
                    ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_float,
                    ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p]
        bwd_args = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                    ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                    ctypes.c_int, ctypes.c_float, ctypes.c_int, ctypes.c_void_p, ctypes.c_size_t,
                    ctypes.c_void_p]
        for name, args in (("roi_align_fpn_forward", fwd_args), ("roi_align_fpn_forward_host", fwd_args),
                           ("roi_align_fpn_backward", bwd_args), ("roi_align_fpn_backward_host", bwd_args)):
            getattr(L, name).restype = ctypes.c_int
            getattr(L, name).argtypes = args
        L.roi_align_fpn_forward_ex.restype = ctypes.c_int
        L.roi_align_fpn_forward_ex.argtypes = fwd_args[:12] + [ctypes.c_int] + fwd_args[12:]
        L.roi_align_fpn_backward_static.restype = ctypes.c_int
        L.roi_align_fpn_backward_static.argtypes = bwd_args[:13] + [ctypes.c_void_p]
        L.roi_align_fpn_backward_ex.restype = ctypes.c_int
        L.roi_align_fpn_backward_ex.argtypes = bwd_args[:3] + [ctypes.c_int] + bwd_args[3:]
        vp, ci, cf = ctypes.c_void_p, ctypes.c_int, ctypes.c_float
        L.roi_pool_fpn_forward.restype = ci
        L.roi_pool_fpn_forward.argtypes = [vp, ci, ci, vp, ci, ci, ci, cf, vp, vp, vp, vp]
        L.roi_pool_fpn_backward.restype = ci
        L.roi_pool_fpn_backward.argtypes = [vp, ci, ci, vp, vp, vp, vp, ci, ci, ci, cf, ci, vp]
        L.roi_deform_pool_fpn_forward.restype = ci
        L.roi_deform_pool_fpn_forward.argtypes = [vp, ci, ci, vp, ci, vp, cf, ci, ci, ci, cf, vp, vp, vp]
        L.roi_deform_pool_fpn_backward.restype = ci
        L.roi_deform_pool_fpn_backward.argtypes = [vp, vp, ci, ci, vp, vp, vp, ci, vp, cf, ci, ci, ci, cf, vp, ci, vp]
        L.roi_align_fc_fpn_forward.restype = ci
        L.roi_align_fc_fpn_forward.argtypes = [vp, ci, ci, vp, ci, ci, ci, ci, ci, cf, vp, vp, ci, vp, vp]
        L.roi_nms_workspace_bytes.restype = ctypes.c_size_t
        L.roi_nms_workspace_bytes.argtypes = [ci]
        L.roi_nms.restype = ci
        L.roi_nms.argtypes = [vp, vp, ci, cf, vp, vp, vp, ctypes.c_size_t, vp]
        L.roi_soft_nms.restype = ci
        L.roi_soft_nms.argtypes = [vp, vp, ci, cf, cf, cf, ci, vp, vp, vp, vp, ctypes.c_size_t, vp]
        L.roi_align_fpn_strerror.restype = ctypes.c_char_p
        L.roi_align_fpn_strerror.argtypes = [ctypes.c_int]
        L.roi_align_fpn_launch_count.restype = ctypes.c_uint64
        _lib = L
    return _lib


def strerror(status: int) -> str:
    return lib().roi_align_fpn_strerror(int(status)).decode()


def launch_count() -> int:
    return int(lib().roi_align_fpn_launch_count())


def _stream_ptr(stream: Optional[torch.cuda.Stream]) -> ctypes.c_void_p:
    s = stream if stream is not None else torch.cuda.current_stream()
    return ctypes.c_void_p(s.cuda_stream)


def _ptr(t: Optional[torch.Tensor]) -> ctypes.c_void_p:
    return ctypes.c_void_p(0 if t is None else t.data_ptr())


def make_levels(tensors: Sequence[torch.Tensor], scales: Sequence[float]):
    """Descriptors for logical-[N,C,H,W] tensors of any strides (NCHW or channels-last views)."""
    arr = (RafLevel * len(tensors))()
    for i, (t, s) in enumerate(zip(tensors, scales)):
        assert t.dim() == 4
        arr[i].data = t.data_ptr()
        arr[i].n, arr[i].c, arr[i].h, arr[i].w = t.shape
        arr[i].sn, arr[i].sc, arr[i].sh, arr[i].sw = t.stride()
        arr[i].spatial_scale = float(s)
    return arr


def _strides4(t: torch.Tensor):
    assert t.dim() == 4
    return (ctypes.c_int64 * 4)(*t.stride())


def roi_align_fpn_workspace_bytes(K: int, L: int, out_h: int, out_w: int, sampling_ratio: int,
                                  flags: int = 0) -> int:
    return int(lib().roi_align_fpn_workspace_bytes(K, L, out_h, out_w, sampling_ratio, flags))


def roi_align_fpn_repack_bytes(levels: Sequence[torch.Tensor], scales: Sequence[float], dtype, K: int, out_h: int,
                               out_w: int) -> int:
    """Extra workspace bytes RAF_REPACK needs (append them to roi_align_fpn_workspace_bytes)."""
    desc = make_levels(levels, scales)
    return int(lib().roi_align_fpn_repack_bytes(desc, len(levels), _DTYPES[dtype], K, out_h, out_w))


def roi_fpn_assign_levels(rois: torch.Tensor, L: int, finest_scale: float,
                          levels: Optional[torch.Tensor], counts: Optional[torch.Tensor],
                          perm: Optional[torch.Tensor], ws: Optional[torch.Tensor] = None,
                          stream=None) -> None:
    K = rois.shape[0]
    rc = lib().roi_fpn_assign_levels(_ptr(rois), K, L, finest_scale, _ptr(levels), _ptr(counts),
                                     _ptr(perm), _ptr(ws), 0 if ws is None else ws.numel() * ws.element_size(),
                                     _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_fpn_assign_levels")


def _check_call(levels: Sequence[torch.Tensor], level_dtype, rois: torch.Tensor, roi_tensor: torch.Tensor,
                roi_tensor_dtype, ws: Optional[torch.Tensor], host: bool = False) -> None:
    """What the C ABI cannot see from raw pointers: dtypes, shapes, contiguity of `rois`, devices.
    Raises ValueError before anything is passed down."""
    if len(levels) == 0:
        raise ValueError("no levels")
    if rois.dtype != torch.float32 or rois.dim() != 2 or rois.shape[1] != 5 or not rois.is_contiguous():
        raise ValueError("rois must be a contiguous float32 [K,5] tensor")
    if roi_tensor.dim() != 4 or roi_tensor.shape[0] != rois.shape[0]:
        raise ValueError("out / grad_out must be logical [K,C,PH,PW] with K = rois.shape[0]")
    if roi_tensor.dtype != roi_tensor_dtype:
        raise ValueError(f"out / grad_out dtype {roi_tensor.dtype} does not match {roi_tensor_dtype}")
    for t in levels:
        if t.dim() != 4 or t.dtype != level_dtype:
            raise ValueError(f"every level must be a 4-d {level_dtype} tensor")
        if t.shape[0] != levels[0].shape[0] or t.shape[1] != levels[0].shape[1]:
            raise ValueError("N and C must be identical across levels")
    if roi_tensor.shape[1] != levels[0].shape[1]:
        raise ValueError("out / grad_out channel count differs from the levels'")
    tensors = list(levels) + [rois, roi_tensor] + ([ws] if ws is not None and not host else [])
    if host:
        if any(t.is_cuda for t in tensors):
            raise ValueError("the *_host entry points take host tensors")
        if ws is None or not ws.is_cuda:
            raise ValueError("arena must be a CUDA tensor")
    else:
        if not all(t.is_cuda for t in tensors) or len({t.device for t in tensors}) != 1:
            raise ValueError("all tensors must live on the same CUDA device")


def roi_align_fpn_forward_ex(feats: Sequence[torch.Tensor], scales: Sequence[float], rois: torch.Tensor,
                             out: torch.Tensor, sampling_ratio: int, aligned: bool, finest_scale: float,
                             flags: int, ws: Optional[torch.Tensor], stream=None, levels_desc=None) -> None:
    """out: logical [K,C,PH,PW] tensor of any strides (e.g. a permuted view of a [K,PH,PW,C] buffer).
    flags: 0 or RAF_NO_PREP (forward only: `ws` may be None)."""
    _check_call(feats, feats[0].dtype if len(feats) else None, rois, out, feats[0].dtype if len(feats) else None, ws)
    if feats[0].dtype not in _DTYPES:
        raise ValueError(f"unsupported feature dtype {feats[0].dtype}")
    desc = levels_desc if levels_desc is not None else make_levels(feats, scales)
    K, _, PH, PW = out.shape
    rc = lib().roi_align_fpn_forward_ex(desc, len(feats), _DTYPES[feats[0].dtype], _ptr(rois), K, PH, PW,
                                        sampling_ratio, int(bool(aligned)), finest_scale, _ptr(out),
                                        _strides4(out), int(flags), _ptr(ws),
                                        0 if ws is None else ws.numel() * ws.element_size(), _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_align_fpn_forward_ex")


def roi_align_fpn_forward(feats: Sequence[torch.Tensor], scales: Sequence[float], rois: torch.Tensor,
                          out: torch.Tensor, sampling_ratio: int, aligned: bool, finest_scale: float,
                          ws: torch.Tensor, stream=None, levels_desc=None) -> None:
    """out: logical [K,C,PH,PW] tensor of any strides (e.g. a permuted view of a [K,PH,PW,C] buffer)."""
    _check_call(feats, feats[0].dtype if len(feats) else None, rois, out, feats[0].dtype if len(feats) else None, ws)
    if feats[0].dtype not in _DTYPES:
        raise ValueError(f"unsupported feature dtype {feats[0].dtype}")
    desc = levels_desc if levels_desc is not None else make_levels(feats, scales)
    K, _, PH, PW = out.shape
    rc = lib().roi_align_fpn_forward(desc, len(feats), _DTYPES[feats[0].dtype], _ptr(rois), K, PH, PW,
                                     sampling_ratio, int(bool(aligned)), finest_scale, _ptr(out),
                                     _strides4(out), _ptr(ws), 0 if ws is None else ws.numel() * ws.element_size(),
                                     _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_align_fpn_forward")


def roi_align_fpn_backward(grad_feats: Sequence[torch.Tensor], scales: Sequence[float],
                           grad_out: torch.Tensor, rois: torch.Tensor, sampling_ratio: int,
                           aligned: bool, finest_scale: float, flags: int, ws: torch.Tensor,
                           stream=None, levels_desc=None) -> None:
    """grad_feats: float32 tensors, or (roi_align_fpn_backward_ex) tensors of grad_out's 16-bit dtype."""
    if grad_out.dtype not in _DTYPES:
        raise ValueError(f"unsupported grad_out dtype {grad_out.dtype}")
    gdt = grad_feats[0].dtype if len(grad_feats) else torch.float32
    if gdt not in (torch.float32, grad_out.dtype):
        raise ValueError("the gradient pyramid must be float32 or have the dtype of grad_out")
    _check_call(grad_feats, gdt, rois, grad_out, grad_out.dtype, ws)
    desc = levels_desc if levels_desc is not None else make_levels(grad_feats, scales)
    K, _, PH, PW = grad_out.shape
    rc = lib().roi_align_fpn_backward_ex(desc, len(grad_feats), _DTYPES[grad_out.dtype], _DTYPES[gdt], _ptr(grad_out),
                                         _strides4(grad_out), _ptr(rois), K, PH, PW, sampling_ratio,
                                         int(bool(aligned)), finest_scale, flags, _ptr(ws),
                                         ws.numel() * ws.element_size(), _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_align_fpn_backward")


RAF_STATIC_WS_BYTES = 4 << 20


def roi_align_fpn_backward_static(grad_feats: Sequence[torch.Tensor], scales: Sequence[float],
                                  grad_out: torch.Tensor, rois: torch.Tensor, sampling_ratio: int,
                                  aligned: bool, finest_scale: float, flags: int = 0, stream=None) -> None:
    """roi_align_fpn_backward without a workspace: the library's static scratch array (RAF_STATIC_WS_BYTES) is used
    and nothing is allocated.  Calls that overlap on the GPU race on that array (include/raf.h)."""
    if grad_out.dtype not in _DTYPES:
        raise ValueError(f"unsupported grad_out dtype {grad_out.dtype}")
    _check_call(grad_feats, torch.float32, rois, grad_out, grad_out.dtype, None)
    K, _, PH, PW = grad_out.shape
    rc = lib().roi_align_fpn_backward_static(make_levels(grad_feats, scales), len(grad_feats), _DTYPES[grad_out.dtype],
                                             _ptr(grad_out), _strides4(grad_out), _ptr(rois), K, PH, PW, sampling_ratio,
                                             int(bool(aligned)), finest_scale, int(flags), _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_align_fpn_backward_static")


def roi_align_fpn_host_arena_bytes(levels: Sequence[torch.Tensor], scales, dtype: torch.dtype, K: int,
                                   out_h: int, out_w: int, sampling_ratio: int, flags: int = 0) -> int:
    desc = make_levels(levels, scales)
    return int(lib().roi_align_fpn_host_arena_bytes(desc, len(levels), _DTYPES[dtype], K, out_h, out_w,
                                                    sampling_ratio, flags))


def roi_align_fpn_forward_host(feats_host: Sequence[torch.Tensor], scales, rois_host: torch.Tensor,
                               out_host: torch.Tensor, sampling_ratio: int, aligned: bool,
                               finest_scale: float, arena: torch.Tensor, stream=None) -> None:
    """HOST (pinned) tensors in and out; `arena` is a device byte buffer."""
    _check_call(feats_host, feats_host[0].dtype if len(feats_host) else None, rois_host, out_host,
                feats_host[0].dtype if len(feats_host) else None, arena, host=True)
    desc = make_levels(feats_host, scales)
    K, _, PH, PW = out_host.shape
    rc = lib().roi_align_fpn_forward_host(desc, len(feats_host), _DTYPES[feats_host[0].dtype],
                                          _ptr(rois_host), K, PH, PW, sampling_ratio, int(bool(aligned)),
                                          finest_scale, _ptr(out_host), _strides4(out_host), _ptr(arena),
                                          arena.numel() * arena.element_size(), _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_align_fpn_forward_host")


def roi_align_fpn_backward_host(grad_feats_host: Sequence[torch.Tensor], scales,
                                grad_out_host: torch.Tensor, rois_host: torch.Tensor,
                                sampling_ratio: int, aligned: bool, finest_scale: float, flags: int,
                                arena: torch.Tensor, stream=None) -> None:
    _check_call(grad_feats_host, torch.float32, rois_host, grad_out_host, grad_out_host.dtype, arena, host=True)
    desc = make_levels(grad_feats_host, scales)
    K, _, PH, PW = grad_out_host.shape
    rc = lib().roi_align_fpn_backward_host(desc, len(grad_feats_host), _DTYPES[grad_out_host.dtype],
                                           _ptr(grad_out_host), _strides4(grad_out_host), _ptr(rois_host),
                                           K, PH, PW, sampling_ratio, int(bool(aligned)), finest_scale,
                                           flags, _ptr(arena), arena.numel() * arena.element_size(),
                                           _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_align_fpn_backward_host")


# ---- RoIPool-max, NMS, Soft-NMS -------------------------------------------------------------
def roi_pool_fpn_forward(feats: Sequence[torch.Tensor], scales: Sequence[float], rois: torch.Tensor,
                         out: torch.Tensor, argmax: Optional[torch.Tensor], finest_scale: float, stream=None) -> None:
    """out: logical [K,C,PH,PW]; argmax: int32 tensor of the same shape AND strides as `out` (or None)."""
    _check_call(feats, feats[0].dtype if len(feats) else None, rois, out, feats[0].dtype if len(feats) else None, None)
    if feats[0].dtype not in _DTYPES:
        raise ValueError(f"unsupported feature dtype {feats[0].dtype}")
    if argmax is not None and (argmax.dtype != torch.int32 or argmax.shape != out.shape or argmax.stride() != out.stride()
                               or argmax.device != out.device):
        raise ValueError("argmax must be an int32 tensor with the shape, strides and device of out")
    K, _, PH, PW = out.shape
    rc = lib().roi_pool_fpn_forward(make_levels(feats, scales), len(feats), _DTYPES[feats[0].dtype], _ptr(rois), K, PH, PW,
                                    finest_scale, _ptr(out), _ptr(argmax), _strides4(out), _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_pool_fpn_forward")


def roi_pool_fpn_backward(grad_feats: Sequence[torch.Tensor], scales: Sequence[float], grad_out: torch.Tensor,
                          argmax: torch.Tensor, rois: torch.Tensor, finest_scale: float, flags: int = 0, stream=None) -> None:
    if grad_out.dtype not in _DTYPES:
        raise ValueError(f"unsupported grad_out dtype {grad_out.dtype}")
    _check_call(grad_feats, torch.float32, rois, grad_out, grad_out.dtype, None)
    if (argmax.dtype != torch.int32 or argmax.shape != grad_out.shape or argmax.stride() != grad_out.stride()
            or argmax.device != grad_out.device):
        raise ValueError("argmax must be an int32 tensor with the shape, strides and device of grad_out")
    K, _, PH, PW = grad_out.shape
    rc = lib().roi_pool_fpn_backward(make_levels(grad_feats, scales), len(grad_feats), _DTYPES[grad_out.dtype], _ptr(grad_out),
                                     _ptr(argmax), _strides4(grad_out), _ptr(rois), K, PH, PW, finest_scale, int(flags),
                                     _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_pool_fpn_backward")


def _check_offset(offset: Optional[torch.Tensor], K: int, PH: int, PW: int, device, what: str) -> None:
    if offset is None:
        return
    if (offset.dtype != torch.float32 or tuple(offset.shape) != (K, 2, PH, PW) or not offset.is_contiguous()
            or offset.device != device):
        raise ValueError(f"{what} must be a contiguous float32 [K,2,PH,PW] tensor on the device of the RoI tensor")


def roi_deform_pool_fpn_forward(feats: Sequence[torch.Tensor], scales: Sequence[float], rois: torch.Tensor,
                                offset: Optional[torch.Tensor], gamma: float, out: torch.Tensor, sampling_ratio: int,
                                finest_scale: float, stream=None) -> None:
    """Deformable RoI pooling (include/raf.h).  out: logical [K,C,PH,PW]; offset: float32 [K,2,PH,PW] or None."""
    _check_call(feats, feats[0].dtype if len(feats) else None, rois, out, feats[0].dtype if len(feats) else None, None)
    if feats[0].dtype not in _DTYPES:
        raise ValueError(f"unsupported feature dtype {feats[0].dtype}")
    K, _, PH, PW = out.shape
    _check_offset(offset, K, PH, PW, out.device, "offset")
    rc = lib().roi_deform_pool_fpn_forward(make_levels(feats, scales), len(feats), _DTYPES[feats[0].dtype], _ptr(rois), K,
                                           _ptr(offset), float(gamma), PH, PW, int(sampling_ratio), finest_scale, _ptr(out),
                                           _strides4(out), _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_deform_pool_fpn_forward")


def roi_deform_pool_fpn_backward(feats: Sequence[torch.Tensor], grad_feats: Optional[Sequence[torch.Tensor]],
                                 scales: Sequence[float], grad_out: torch.Tensor, rois: torch.Tensor,
                                 offset: Optional[torch.Tensor], gamma: float, sampling_ratio: int, finest_scale: float,
                                 grad_offset: Optional[torch.Tensor], flags: int = 0, stream=None) -> None:
    """grad_feats: fp32 tensors shaped like feats (or None); grad_offset: float32 [K,2,PH,PW] (or None)."""
    if grad_out.dtype not in _DTYPES:
        raise ValueError(f"unsupported grad_out dtype {grad_out.dtype}")
    _check_call(feats, grad_out.dtype, rois, grad_out, grad_out.dtype, None)
    if grad_feats is not None:
        _check_call(grad_feats, torch.float32, rois, grad_out, grad_out.dtype, None)
        if any(tuple(g.shape) != tuple(f.shape) for g, f in zip(grad_feats, feats)) or len(grad_feats) != len(feats):
            raise ValueError("grad_feats must have the shapes of feats")
    K, _, PH, PW = grad_out.shape
    _check_offset(offset, K, PH, PW, grad_out.device, "offset")
    _check_offset(grad_offset, K, PH, PW, grad_out.device, "grad_offset")
    rc = lib().roi_deform_pool_fpn_backward(make_levels(feats, scales),
                                            None if grad_feats is None else make_levels(grad_feats, scales), len(feats),
                                            _DTYPES[grad_out.dtype], _ptr(grad_out), _strides4(grad_out), _ptr(rois), K,
                                            _ptr(offset), float(gamma), PH, PW, int(sampling_ratio), finest_scale,
                                            _ptr(grad_offset), int(flags), _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_deform_pool_fpn_backward")


def roi_align_fc_fpn_forward(feats: Sequence[torch.Tensor], scales: Sequence[float], rois: torch.Tensor,
                             weight: torch.Tensor, bias: Optional[torch.Tensor], out: torch.Tensor, out_size,
                             sampling_ratio: int, aligned: bool, finest_scale: float, stream=None) -> None:
    """RoIAlign gather fused into the first FC (include/raf.h).  weight: [n_out, PH*PW*C] in the feature dtype, columns in
    (ph, pw, c) order; bias: float32 [n_out] or None; out: float32 [K, n_out] contiguous."""
    if len(feats) == 0 or feats[0].dtype not in _DTYPES:
        raise ValueError("unsupported feature dtype")
    PH, PW = out_size
    K, C = rois.shape[0], feats[0].shape[1]
    if rois.dtype != torch.float32 or rois.dim() != 2 or rois.shape[1] != 5 or not rois.is_contiguous():
        raise ValueError("rois must be a contiguous float32 [K,5] tensor")
    if (weight.dtype != feats[0].dtype or weight.dim() != 2 or weight.shape[1] != PH * PW * C or not weight.is_contiguous()):
        raise ValueError("weight must be a contiguous [n_out, PH*PW*C] tensor of the feature dtype")
    n_out = weight.shape[0]
    if bias is not None and (bias.dtype != torch.float32 or tuple(bias.shape) != (n_out,) or not bias.is_contiguous()):
        raise ValueError("bias must be a contiguous float32 [n_out] tensor")
    if out.dtype != torch.float32 or tuple(out.shape) != (K, n_out) or not out.is_contiguous():
        raise ValueError("out must be a contiguous float32 [K, n_out] tensor")
    tensors = list(feats) + [rois, weight, out] + ([bias] if bias is not None else [])
    if not all(t.is_cuda for t in tensors) or len({t.device for t in tensors}) != 1:
        raise ValueError("all tensors must live on the same CUDA device")
    rc = lib().roi_align_fc_fpn_forward(make_levels(feats, scales), len(feats), _DTYPES[feats[0].dtype], _ptr(rois), K, PH, PW,
                                        int(sampling_ratio), int(bool(aligned)), finest_scale, _ptr(weight), _ptr(bias),
                                        n_out, _ptr(out), _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_align_fc_fpn_forward")


def _check_boxes(boxes: torch.Tensor, scores: torch.Tensor) -> int:
    if boxes.dtype != torch.float32 or boxes.dim() != 2 or boxes.shape[1] != 4 or not boxes.is_contiguous():
        raise ValueError("boxes must be a contiguous float32 [n,4] tensor")
    if scores.dtype != torch.float32 or scores.dim() != 1 or scores.shape[0] != boxes.shape[0] or not scores.is_contiguous():
        raise ValueError("scores must be a contiguous float32 [n] tensor")
    if not (boxes.is_cuda and scores.is_cuda and boxes.device == scores.device):
        raise ValueError("boxes and scores must live on the same CUDA device")
    return boxes.shape[0]


def roi_nms_workspace_bytes(n: int) -> int:
    return int(lib().roi_nms_workspace_bytes(int(n)))


def roi_nms(boxes: torch.Tensor, scores: torch.Tensor, iou_threshold: float, keep: torch.Tensor, num_keep: torch.Tensor,
            ws: Optional[torch.Tensor], stream=None) -> None:
    """keep: int32 [n] device, num_keep: int32 [1] device (the caller reads it when it needs the count)."""
    n = _check_boxes(boxes, scores)
    if keep.dtype != torch.int32 or keep.numel() < n or num_keep.dtype != torch.int32 or not keep.is_cuda or not num_keep.is_cuda:
        raise ValueError("keep must be int32 [n] and num_keep int32 [1], on the device")
    rc = lib().roi_nms(_ptr(boxes), _ptr(scores), n, float(iou_threshold), _ptr(keep), _ptr(num_keep), _ptr(ws),
                       0 if ws is None else ws.numel() * ws.element_size(), _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_nms")


def roi_soft_nms(boxes: torch.Tensor, scores: torch.Tensor, iou_threshold: float, sigma: float, min_score: float,
                 method: int, keep: torch.Tensor, new_scores: torch.Tensor, num_keep: torch.Tensor, stream=None) -> None:
    n = _check_boxes(boxes, scores)
    if (keep.dtype != torch.int32 or keep.numel() < n or new_scores.dtype != torch.float32 or new_scores.numel() < n
            or num_keep.dtype != torch.int32 or not (keep.is_cuda and new_scores.is_cuda and num_keep.is_cuda)):
        raise ValueError("keep int32 [n], new_scores float32 [n], num_keep int32 [1], on the device")
    rc = lib().roi_soft_nms(_ptr(boxes), _ptr(scores), n, float(iou_threshold), float(sigma), float(min_score), int(method),
                            _ptr(keep), _ptr(new_scores), _ptr(num_keep), None, 0, _stream_ptr(stream))
    if rc:
        raise RafError(rc, "roi_soft_nms")
