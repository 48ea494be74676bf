"""ctypes front end of the CPU oracle for RoIPool-max, NMS, Soft-NMS and deformable RoI pooling (oracle/ops_ref.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the product
package and holds no arithmetic of its own: argument marshalling only (numpy in, numpy out).
"""
import ctypes

import numpy as np

from . import build as _build


class _Level(ctypes.Structure):
    _fields_ = [("data", ctypes.c_void_p), ("n", ctypes.c_int32), ("c", ctypes.c_int32),
                ("h", ctypes.c_int32), ("w", ctypes.c_int32), ("spatial_scale", ctypes.c_float)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build_ops())
        _lib.ops_ref_iou.restype = ctypes.c_float
    return _lib


def _levels(arrays, scales):
    lv = (_Level * len(arrays))()
    for i, (a, s) in enumerate(zip(arrays, scales)):
        assert a.dtype == np.float64 and a.flags.c_contiguous and a.ndim == 4
        lv[i].data = a.ctypes.data
        lv[i].n, lv[i].c, lv[i].h, lv[i].w = a.shape
        lv[i].spatial_scale = float(s)
    return lv


def _p(a):
    return ctypes.c_void_p(a.ctypes.data)


def roi_pool_forward(feats, scales, rois, out_size, finest_scale=56.0):
    """P1-P3.  Returns (out float64 [K,C,PH,PW], argmax int32 [K,C,PH,PW] = y*W + x on the RoI's level, -1: none)."""
    feats64 = [np.ascontiguousarray(f, dtype=np.float64) for f in feats]
    rois = np.ascontiguousarray(rois, dtype=np.float32)
    PH, PW = out_size
    K, C = rois.shape[0], feats64[0].shape[1]
    out = np.zeros((K, C, PH, PW), np.float64)
    arg = np.full((K, C, PH, PW), -1, np.int32)
    rc = lib().roi_pool_fpn_forward_ref(_levels(feats64, scales), len(feats64), _p(rois), K, PH, PW,
                                        ctypes.c_float(finest_scale), _p(out), _p(arg))
    assert rc == 0
    return out, arg


def roi_pool_backward(shapes, scales, grad_out, argmax, rois, finest_scale=56.0, accumulate_into=None):
    """P4.  Returns the list of float64 gradient arrays."""
    rois = np.ascontiguousarray(rois, dtype=np.float32)
    grad_out = np.ascontiguousarray(grad_out, dtype=np.float64)
    argmax = np.ascontiguousarray(argmax, dtype=np.int32)
    K, C, PH, PW = grad_out.shape
    if accumulate_into is not None:
        grads = [np.ascontiguousarray(g, dtype=np.float64).copy() for g in accumulate_into]
    else:
        grads = [np.zeros(s, np.float64) for s in shapes]
    rc = lib().roi_pool_fpn_backward_ref(_levels(grads, scales), len(grads), _p(grad_out), _p(argmax), _p(rois), K,
                                         PH, PW, ctypes.c_float(finest_scale))
    assert rc == 0
    return grads


def iou(a, b):
    a = np.ascontiguousarray(a, dtype=np.float32)
    b = np.ascontiguousarray(b, dtype=np.float32)
    return float(lib().ops_ref_iou(_p(a), _p(b)))


def nms(boxes, scores, iou_threshold):
    """N1-N3.  Kept indices (int32) in descending-score order."""
    boxes = np.ascontiguousarray(boxes, dtype=np.float32)
    scores = np.ascontiguousarray(scores, dtype=np.float32)
    n = boxes.shape[0]
    keep = np.zeros(max(n, 1), np.int32)
    nk = lib().nms_ref(_p(boxes), _p(scores), n, ctypes.c_float(iou_threshold), _p(keep))
    return keep[:nk].copy()


def soft_nms(boxes, scores, iou_threshold, sigma, min_score, method):
    """N4-N6.  method: 'linear' | 'gaussian'.  Returns (indices int32, rescored float32) in selection order."""
    boxes = np.ascontiguousarray(boxes, dtype=np.float32)
    scores = np.ascontiguousarray(scores, dtype=np.float32)
    n = boxes.shape[0]
    keep = np.zeros(max(n, 1), np.int32)
    ns = np.zeros(max(n, 1), np.float32)
    nk = lib().soft_nms_ref(_p(boxes), _p(scores), n, ctypes.c_float(iou_threshold), ctypes.c_float(sigma),
                            ctypes.c_float(min_score), {"linear": 1, "gaussian": 2}[method], _p(keep), _p(ns))
    return keep[:nk].copy(), ns[:nk].copy()


def deform_roi_pool_forward(feats, scales, rois, offset, gamma, out_size, sampling_ratio=2, finest_scale=56.0, f64=False):
    """D1-D4.  offset: float32 [K,2,PH,PW] (plane 0 = x, 1 = y) or None.  Returns float64 [K,C,PH,PW]."""
    feats64 = [np.ascontiguousarray(f, dtype=np.float64) for f in feats]
    rois = np.ascontiguousarray(rois, dtype=np.float32)
    PH, PW = out_size
    K, C = rois.shape[0], feats64[0].shape[1]
    off = None if offset is None else np.ascontiguousarray(offset, dtype=np.float32)
    assert off is None or off.shape == (K, 2, PH, PW)
    out = np.zeros((K, C, PH, PW), np.float64)
    rc = lib().deform_roi_pool_fpn_forward_ref(_levels(feats64, scales), len(feats64), _p(rois), K,
                                               None if off is None else _p(off), ctypes.c_float(gamma), PH, PW,
                                               int(sampling_ratio), ctypes.c_float(finest_scale), int(bool(f64)), _p(out))
    assert rc == 0
    return out


def deform_roi_pool_backward(feats, scales, grad_out, rois, offset, gamma, sampling_ratio=2, finest_scale=56.0, f64=False):
    """D5.  Returns (list of float64 feature gradients, float64 offset gradient [K,2,PH,PW])."""
    feats64 = [np.ascontiguousarray(f, dtype=np.float64) for f in feats]
    grads = [np.zeros(f.shape, np.float64) for f in feats64]
    rois = np.ascontiguousarray(rois, dtype=np.float32)
    grad_out = np.ascontiguousarray(grad_out, dtype=np.float64)
    K, C, PH, PW = grad_out.shape
    off = None if offset is None else np.ascontiguousarray(offset, dtype=np.float32)
    goff = np.zeros((K, 2, PH, PW), np.float64)
    rc = lib().deform_roi_pool_fpn_backward_ref(_levels(feats64, scales), _levels(grads, scales), len(feats64), _p(grad_out),
                                                _p(rois), K, None if off is None else _p(off), ctypes.c_float(gamma), PH, PW,
                                                int(sampling_ratio), ctypes.c_float(finest_scale), int(bool(f64)), _p(goff))
    assert rc == 0
    return grads, goff


def _round_to(x64, dtype):
    """float64 -> the value a 16-bit (or fp32) store keeps, returned as float64 (round to nearest even)."""
    if dtype == "f32":
        return x64.astype(np.float32).astype(np.float64)
    if dtype == "f16":
        return x64.astype(np.float16).astype(np.float64)
    assert dtype == "bf16"
    u = x64.astype(np.float32).view(np.uint32).astype(np.uint64)
    u = ((u + 0x7FFF + ((u >> 16) & 1)) >> 16) << 16          # round to nearest even on the upper 16 bits
    return u.astype(np.uint32).view(np.float32).astype(np.float64)


def roi_align_fc_forward(feats, scales, rois, weight, bias, out_size, sampling_ratio, aligned, finest_scale=56.0,
                         dtype="bf16"):
    """RoIExtractor -> first FC of the box head (readings F1-F3), as a composition:
    (1) RoIAlign forward of the pinned oracle (oracle/raf_ref.cpp, spec mode); (2) every feature rounded to `dtype`, as
    the RoI feature tensor the head would read (F2); (3) flattened per RoI in (ph, pw, c) order (F1); (4) a library
    matrix product in float64 with the weight [N_out, PH*PW*C] (+ bias).  Returns float64 [K, N_out]."""
    from . import raf_ref as _raf
    x = _raf.forward(feats, scales, rois, out_size, sampling_ratio, aligned, finest_scale, coord_f32=True)   # [K,C,PH,PW]
    x = _round_to(x, dtype)
    K = x.shape[0]
    a = np.ascontiguousarray(x.transpose(0, 2, 3, 1)).reshape(K, -1)                                            # (ph, pw, c)
    w = np.ascontiguousarray(weight, dtype=np.float64)
    assert w.shape[1] == a.shape[1]
    out = a @ w.T
    if bias is not None:
        out = out + np.asarray(bias, dtype=np.float64)[None, :]
    return out
