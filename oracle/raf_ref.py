"""ctypes front end of the CPU oracle (oracle/raf_ref.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the product
package and holds no arithmetic of its own: argument marshalling only (numpy in, numpy out).
"""
import ctypes
import os

import numpy as np

from . import build as _build


class _Level(ctypes.Structure):
    _fields_ = [("data", ctypes.c_void_p), ("n", ctypes.c_int32), ("c", ctypes.c_int32),
                ("h", ctypes.c_int32), ("w", ctypes.c_int32), ("spatial_scale", ctypes.c_float)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        _lib.raf_ref_level_of.restype = ctypes.c_int32
        _lib.raf_ref_level_of.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_float]
        _lib.raf_ref_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(lib().raf_ref_num_threads())


def _rois32(rois):
    rois = np.ascontiguousarray(rois, dtype=np.float32)
    assert rois.ndim == 2 and rois.shape[1] == 5, rois.shape
    return rois


def _level_array(arrays, scales):
    lv = (_Level * len(arrays))()
    for i, (a, s) in enumerate(zip(arrays, scales)):
        assert a.dtype == np.float64 and a.flags.c_contiguous and a.ndim == 4
        lv[i].data = a.ctypes.data
        lv[i].n, lv[i].c, lv[i].h, lv[i].w = a.shape
        lv[i].spatial_scale = float(s)
    return lv


def assign_levels(rois, L, finest_scale):
    """C1 + C2 -> (levels[K] int32, counts[L] int32, perm[K] int32)."""
    rois = _rois32(rois)
    K = rois.shape[0]
    levels = np.zeros(K, np.int32)
    counts = np.zeros(L, np.int32)
    perm = np.zeros(K, np.int32)
    rc = lib().roi_fpn_assign_levels_ref(
        ctypes.c_void_p(rois.ctypes.data), K, L, ctypes.c_float(finest_scale),
        ctypes.c_void_p(levels.ctypes.data), ctypes.c_void_p(counts.ctypes.data),
        ctypes.c_void_p(perm.ctypes.data))
    assert rc == 0, rc
    return levels, counts, perm


def forward(feats, scales, rois, out_size, sampling_ratio, aligned, finest_scale=56.0,
            coord_f32=True):
    """C3 + C5.  feats: list of [N,C,H_l,W_l] arrays (widened exactly to float64).
    Returns float64 [K,C,PH,PW], un-rounded."""
    feats64 = [np.ascontiguousarray(f, dtype=np.float64) for f in feats]
    rois = _rois32(rois)
    PH, PW = out_size
    K, C = rois.shape[0], feats64[0].shape[1]
    out = np.zeros((K, C, PH, PW), np.float64)
    lv = _level_array(feats64, scales)
    rc = lib().roi_align_fpn_forward_ref(
        lv, len(feats64), ctypes.c_void_p(rois.ctypes.data), K, PH, PW, int(sampling_ratio),
        int(bool(aligned)), ctypes.c_float(finest_scale), int(bool(coord_f32)),
        ctypes.c_void_p(out.ctypes.data))
    assert rc == 0, rc
    return out


def backward(shapes, scales, grad_out, rois, out_size, sampling_ratio, aligned,
             finest_scale=56.0, coord_f32=True, accumulate_into=None, want_abs_sum=True):
    """C4.  shapes: list of (N,C,H_l,W_l).  Returns (grads, S): lists of float64 arrays;
    S[l] = sum |w * gout / count| per element (tolerance scale, reading S11) or None."""
    rois = _rois32(rois)
    PH, PW = out_size
    K = rois.shape[0]
    grad_out = np.ascontiguousarray(grad_out, dtype=np.float64)
    assert grad_out.shape == (K, shapes[0][1], PH, PW), grad_out.shape
    if accumulate_into is not None:
        grads = [np.ascontiguousarray(g, dtype=np.float64).copy() for g in accumulate_into]
    else:
        grads = [np.zeros(s, np.float64) for s in shapes]
    S = [np.zeros(s, np.float64) for s in shapes] if want_abs_sum else None
    lv = _level_array(grads, scales)
    if S is not None:
        sp = (ctypes.c_void_p * len(S))(*[s.ctypes.data for s in S])
    else:
        sp = None
    rc = lib().roi_align_fpn_backward_ref(
        lv, sp, len(grads), ctypes.c_void_p(grad_out.ctypes.data),
        ctypes.c_void_p(rois.ctypes.data), K, PH, PW, int(sampling_ratio), int(bool(aligned)),
        ctypes.c_float(finest_scale), int(bool(coord_f32)), int(accumulate_into is not None))
    assert rc == 0, rc
    return grads, S


def footprint(shapes, scales, rois, out_size, sampling_ratio, aligned, finest_scale=56.0):
    """Union of touched pixels (SURVEY 8(d) `U`): list of uint8 masks [N,H_l,W_l]."""
    rois = _rois32(rois)
    PH, PW = out_size
    masks = [np.zeros((s[0], s[2], s[3]), np.uint8) for s in shapes]
    dummy = [np.zeros((1, 1, 1, 1), np.float64) for _ in shapes]
    lv = _level_array(dummy, scales)
    for i, s in enumerate(shapes):
        lv[i].n, lv[i].c, lv[i].h, lv[i].w = s
    mp = (ctypes.c_void_p * len(masks))(*[m.ctypes.data for m in masks])
    rc = lib().roi_align_fpn_footprint_ref(
        mp, lv, len(masks), ctypes.c_void_p(rois.ctypes.data), rois.shape[0], PH, PW,
        int(sampling_ratio), int(bool(aligned)), ctypes.c_float(finest_scale))
    assert rc == 0, rc
    return masks
