"""Algorithmic-byte accounting for the roofline lines of bench.py.

Host-side measurement helper (numpy), not part of the compute path and not shared with the oracle:
it enumerates which pyramid pixels a RoI set touches so that the forward's compulsory read set is
the UNION of touched pixels, not the dense pyramid and not the 4*g^2*P^2 requested taps.

  forward   B_f = U*C*s_feat + K*C*PH*PW*s_out + 20*K
  backward  B_b = K*C*PH*PW*s_gout + (sum_l N*C*H_l*W_l)*4          (overwrite mode)
            B_b = K*C*PH*PW*s_gout + 2*U*C*4                         (accumulate mode)
"""
from typing import Dict, List, Sequence, Tuple

import numpy as np

f32 = np.float32


def _levels_f32(rois: np.ndarray, L: int, finest_scale: float) -> np.ndarray:
    w = rois[:, 3] - rois[:, 1]
    h = rois[:, 4] - rois[:, 2]
    with np.errstate(invalid="ignore"):
        t = np.sqrt(w * h) / f32(finest_scale) + f32(1e-6)
    lv = np.zeros(len(rois), np.int64)
    for j in range(1, L):
        lv += (t >= f32(2.0 ** j))
    return lv


def _axis_pixels(start: np.float32, extent_end: np.float32, P: int, g: int, n: int, aligned: bool):
    """Touched pixel indices along one axis + number of valid samples (fp32 step by step)."""
    off = f32(0.5) if aligned else f32(0.0)
    s = f32(start - off)
    e = f32(extent_end - off)
    r = f32(e - s)
    if not aligned:
        r = max(r, f32(1.0))
    b = f32(r / f32(P))
    p = np.repeat(np.arange(P, dtype=f32), g)
    i = np.tile(np.arange(g, dtype=f32), P)
    v = (s + p * b).astype(f32) + ((i + f32(0.5)) * b).astype(f32) / f32(g)
    v = v.astype(f32)
    valid = (v >= -1) & (v <= n)
    v = np.maximum(v[valid], 0)
    lo = np.minimum(v.astype(np.int64), n - 1)
    hi = np.minimum(lo + 1, n - 1)
    return np.unique(np.concatenate([lo, hi])), int(valid.sum())


def footprint(rois: np.ndarray, level_shapes: Sequence[Tuple[int, int, int, int]], scales: Sequence[float],
              out_size: Tuple[int, int], sampling_ratio: int, aligned: bool, finest_scale: float) -> Dict:
    """Union / per-RoI / requested pixel counts for a RoI set (sampling_ratio > 0)."""
    assert sampling_ratio > 0
    rois = np.ascontiguousarray(rois, f32)
    L = len(level_shapes)
    N = level_shapes[0][0]
    PH, PW = out_size
    lv = _levels_f32(rois, L, finest_scale)
    masks = [np.zeros((s[0], s[2], s[3]), bool) for s in level_shapes]
    per_roi = 0
    requested = 0
    for k in range(len(rois)):
        b = rois[k, 0]
        if not (0 <= b < N) or int(b) != b:
            continue
        l = int(lv[k])
        sc = f32(scales[l])
        H, W = level_shapes[l][2], level_shapes[l][3]
        rows, vy = _axis_pixels(f32(rois[k, 2] * sc), f32(rois[k, 4] * sc), PH, sampling_ratio, H, aligned)
        cols, vx = _axis_pixels(f32(rois[k, 1] * sc), f32(rois[k, 3] * sc), PW, sampling_ratio, W, aligned)
        per_roi += len(rows) * len(cols)
        requested += vy * vx * 4
        if len(rows) and len(cols):
            masks[l][int(b)][np.ix_(rows, cols)] = True
    return {"union_px": int(sum(m.sum() for m in masks)), "per_roi_px": int(per_roi),
            "requested_px": int(requested), "pyramid_px": int(sum(s[0] * s[2] * s[3] for s in level_shapes)),
            "level_hist": np.bincount(lv, minlength=L).tolist()}


def algorithmic_bytes(fp: Dict, K: int, C: int, out_size: Tuple[int, int], feat_bytes: int, out_bytes: int,
                      gout_bytes: int, accumulate: bool = False, grad_bytes: int = 4) -> Dict[str, int]:
    PH, PW = out_size
    out_elems = K * C * PH * PW
    fwd = fp["union_px"] * C * feat_bytes + out_elems * out_bytes + 20 * K
    if accumulate:
        bwd = out_elems * gout_bytes + 2 * fp["union_px"] * C * grad_bytes
    else:
        bwd = out_elems * gout_bytes + fp["pyramid_px"] * C * grad_bytes
    return {"fwd": int(fwd), "bwd": int(bwd), "requested_fwd": int(fp["requested_px"] * C * feat_bytes),
            "per_roi_fwd": int(fp["per_roi_px"] * C * feat_bytes)}
