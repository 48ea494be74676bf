"""Pins of the CPU oracle for RoIPool-max, NMS and Soft-NMS (oracle/ops_ref.cpp, readings
P1-P4 / N1-N6 of DESIGN.md 3b).  Nothing here touches the CUDA path; all -m "not gpu"."""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import ops_ref as O


# ------------------------------------------------------------------------------------------ RoIPool-max
def _ramp(H, W, C=1, N=1):
    f = (np.arange(H)[:, None] * W + np.arange(W)[None, :]).astype(np.float64)
    return np.broadcast_to(f, (N, C, H, W)).copy()


def _windows_exact(lo, hi, P, n):
    """Bin windows of an INTEGER extent [lo, hi] (scale 1) in exact rational arithmetic."""
    size = max(hi - lo + 1, 1)
    b = Fraction(size, P)
    out = []
    for p in range(P):
        s = math.floor(p * b) + lo
        e = math.ceil((p + 1) * b) + lo
        out.append((min(max(s, 0), n), min(max(e, 0), n)))
    return out


def test_roi_pool_integer_aligned_identity_and_block_max():
    H = W = 16
    f = _ramp(H, W)
    # 7x7 pixels, 7x7 bins: every bin is one pixel -> identity crop
    out, arg = O.roi_pool_forward([f], [1.0], np.array([[0, 2, 3, 8, 9]], np.float32), (7, 7))
    assert np.array_equal(out[0, 0], f[0, 0, 3:10, 2:9])
    assert np.array_equal(arg[0, 0], (np.arange(3, 10)[:, None] * W + np.arange(2, 9)[None, :]))
    # 14x14 pixels, 7x7 bins: 2x2 blocks, max of an increasing ramp = bottom-right pixel of the block
    out, arg = O.roi_pool_forward([f], [1.0], np.array([[0, 0, 0, 13, 13]], np.float32), (7, 7))
    assert np.array_equal(out[0, 0], f[0, 0, 1:14:2, 1:14:2])
    # on the negated ramp the FIRST pixel of the block wins: the window start is pinned too
    out, arg = O.roi_pool_forward([-f], [1.0], np.array([[0, 0, 0, 13, 13]], np.float32), (7, 7))
    assert np.array_equal(out[0, 0], -f[0, 0, 0:14:2, 0:14:2])


def test_roi_pool_windows_match_exact_rational_arithmetic():
    """Random integer boxes (scale 1, so quantisation is exact): the window of every bin, read back from the
    argmax on an increasing ramp (last pixel) and on a decreasing ramp (first pixel), equals the window
    computed with exact fractions -- including boxes partly or wholly outside the map and empty bins."""
    rng = np.random.default_rng(7)
    H, W = 20, 24
    f = _ramp(H, W)
    for P in ((7, 7), (3, 5), (14, 14)):
        for _ in range(60):
            x1, y1 = int(rng.integers(-6, W)), int(rng.integers(-6, H))
            x2, y2 = x1 + int(rng.integers(0, 22)), y1 + int(rng.integers(0, 22))
            roi = np.array([[0, x1, y1, x2, y2]], np.float32)
            up, au = O.roi_pool_forward([f], [1.0], roi, P)
            dn, ad = O.roi_pool_forward([-f], [1.0], roi, P)
            wy = _windows_exact(y1, y2, P[0], H)
            wx = _windows_exact(x1, x2, P[1], W)
            for ph, (hs, he) in enumerate(wy):
                for pw, (ws, we) in enumerate(wx):
                    if he <= hs or we <= ws:
                        assert au[0, 0, ph, pw] == -1 and up[0, 0, ph, pw] == 0.0
                    else:
                        assert au[0, 0, ph, pw] == (he - 1) * W + (we - 1)
                        assert ad[0, 0, ph, pw] == hs * W + ws
                        assert up[0, 0, ph, pw] == f[0, 0, he - 1, we - 1]


def test_roi_pool_rounding_of_scaled_corners():
    """roundf (half away from zero) of x*scale decides the window: 2.5 -> 3, 3.49 -> 3, -0.5 -> -1."""
    f = _ramp(12, 12)
    # scale 0.25: x1 = 10 -> 2.5 -> 3 ; x2 = 22 -> 5.5 -> 6 ; one bin -> whole window [3, 6]
    out, arg = O.roi_pool_forward([-f], [0.25], np.array([[0, 10, 10, 22, 22]], np.float32), (1, 1))
    assert arg[0, 0, 0, 0] == 3 * 12 + 3
    out, arg = O.roi_pool_forward([f], [0.25], np.array([[0, 10, 10, 22, 22]], np.float32), (1, 1))
    assert arg[0, 0, 0, 0] == 6 * 12 + 6
    out, arg = O.roi_pool_forward([-f], [0.25], np.array([[0, 13.96, 13.96, 22, 22]], np.float32), (1, 1))
    assert arg[0, 0, 0, 0] == 3 * 12 + 3          # 3.49 -> 3
    out, arg = O.roi_pool_forward([-f], [1.0], np.array([[0, -0.5, -0.5, 3, 3]], np.float32), (1, 1))
    assert arg[0, 0, 0, 0] == 0                    # -0.5 -> -1, clamped to 0


def test_roi_pool_constant_ties_invalid_and_levels():
    c = np.full((2, 3, 8, 8), 2.5)
    out, arg = O.roi_pool_forward([c], [1.0], np.array([[1, 1, 1, 5, 6], [7, 1, 1, 5, 6], [0.5, 1, 1, 5, 6]], np.float32), (3, 3))
    assert np.all(out[0] == 2.5) and np.all(out[1:] == 0) and np.all(arg[1:] == -1)
    # ties: the FIRST maximum in row-major order
    assert arg[0, 0, 0, 0] == 1 * 8 + 1
    # NaN never wins; an all-NaN window yields 0 / -1
    d = c.copy(); d[0, 0, 2, 2] = np.nan
    out, arg = O.roi_pool_forward([d], [1.0], np.array([[0, 2, 2, 2, 2]], np.float32), (1, 1))
    assert out[0, 0, 0, 0] == 0 and arg[0, 0, 0, 0] == -1 and out[0, 1, 0, 0] == 2.5
    # level routing: side 50 -> level 0 (scale 1/4), side 300 -> level 2 (scale 1/16), finest_scale 56
    feats = [np.full((1, 1, 64, 64), float(l)) for l in range(4)]
    scales = [1 / 4, 1 / 8, 1 / 16, 1 / 32]
    out, _ = O.roi_pool_forward(feats, scales, np.array([[0, 10, 10, 60, 60], [0, 10, 10, 310, 310]], np.float32), (2, 2))
    assert np.all(out[0] == 0.0) and np.all(out[1] == 2.0)


def test_roi_pool_matches_library_routine():
    tv = pytest.importorskip("torchvision")
    import torch
    rng = np.random.default_rng(11)
    for scale, P in ((1.0, (7, 7)), (0.25, (7, 7)), (0.5, (3, 5))):
        f = rng.standard_normal((2, 3, 24, 30))
        K = 60
        x1 = rng.uniform(-5, 30 / scale, K); y1 = rng.uniform(-5, 24 / scale, K)
        w = rng.uniform(0, 25 / scale, K); h = rng.uniform(0, 25 / scale, K)
        rois = np.stack([rng.integers(0, 2, K), x1, y1, x1 + w, y1 + h], 1).astype(np.float32)
        out, _ = O.roi_pool_forward([f], [scale], rois, P, finest_scale=1e9)
        ref = tv.ops.roi_pool(torch.from_numpy(f), torch.from_numpy(rois).double(), P, scale).numpy()
        assert np.array_equal(out, ref)


def test_roi_pool_backward_is_the_transpose_of_the_selection():
    rng = np.random.default_rng(5)
    shapes = [(2, 3, 20, 28), (2, 3, 10, 14)]
    feats = [rng.standard_normal(s) for s in shapes]
    scales = [0.25, 0.125]
    K = 40
    side = np.exp(rng.uniform(np.log(8), np.log(200), K))
    cx, cy = rng.uniform(0, 112, K), rng.uniform(0, 80, K)
    rois = np.stack([rng.integers(0, 2, K), cx - side / 2, cy - side / 2, cx + side / 2, cy + side / 2], 1).astype(np.float32)
    out, arg = O.roi_pool_forward(feats, scales, rois, (7, 7))
    g = rng.standard_normal(out.shape)
    grads = O.roi_pool_backward(shapes, scales, g, arg, rois)
    # <pool(x), g> = <x, pool^T g> (the forward is x[argmax])
    lhs = float((out * g).sum())
    rhs = float(sum((f * gr).sum() for f, gr in zip(feats, grads)))
    assert abs(lhs - rhs) <= 1e-12 * max(1.0, abs(lhs))
    # mass: every valid bin delivers its gradient exactly once
    assert abs(sum(gr.sum() for gr in grads) - g[arg >= 0].sum()) < 1e-10
    # brute force with numpy scatter
    from oracle import raf_ref as R
    lv = R.assign_levels(rois, 2, 56.0)[0]
    want = [np.zeros(s) for s in shapes]
    for k in range(K):
        b = int(rois[k, 0])
        flat = want[lv[k]][b].reshape(3, -1)
        for c in range(3):
            m = arg[k, c] >= 0
            np.add.at(flat[c], arg[k, c][m], g[k, c][m])
    for a_, b_ in zip(grads, want):
        assert np.allclose(a_, b_, rtol=0, atol=1e-12)


# ---------------------------------------------------------------------------------------------- NMS
def test_iou_closed_forms():
    assert O.iou([0, 0, 2, 2], [0, 0, 2, 2]) == 1.0
    assert O.iou([0, 0, 2, 2], [2, 0, 4, 2]) == 0.0            # touching edges
    assert O.iou([0, 0, 2, 2], [5, 5, 6, 6]) == 0.0
    assert O.iou([0, 0, 4, 4], [1, 1, 3, 3]) == np.float32(4) / np.float32(16)     # contained: area ratio
    assert O.iou([0, 0, 2, 2], [1, 1, 3, 3]) == np.float32(np.float32(1) / np.float32(7))
    assert O.iou([0, 0, 2, 2], [1, 1, 3, 3]) == O.iou([1, 1, 3, 3], [0, 0, 2, 2])
    assert math.isnan(O.iou([1, 1, 1, 1], [1, 1, 1, 1]))       # 0/0: compares false everywhere


def test_nms_worked_example_and_threshold_edge():
    boxes = np.array([[0, 0, 10, 10], [1, 1, 11, 11], [20, 20, 30, 30], [0, 0, 10, 9], [21, 21, 29, 29]], np.float32)
    scores = np.array([0.9, 0.8, 0.7, 0.95, 0.1], np.float32)
    # order: 3, 0, 1, 2, 4.  IoU(3,0) = 90/100 = 0.9 -> 0 out; IoU(3,1) = 72/(90+100-72) = 0.61 -> 1 out;
    # 2 kept; IoU(2,4) = 64/100 = 0.64 -> 4 out at threshold 0.5
    assert O.nms(boxes, scores, 0.5).tolist() == [3, 2]
    assert O.nms(boxes, scores, 0.62).tolist() == [3, 1, 2]      # 0.61 no longer suppresses 1; 0.64 still suppresses 4
    assert O.nms(boxes, scores, 0.65).tolist() == [3, 1, 2, 4]   # (0 stays out: IoU(3,0) = 0.9)
    assert O.nms(boxes, scores, 0.95).tolist() == [3, 0, 1, 2, 4]
    # strict comparison: IoU == threshold is kept
    b = np.array([[0, 0, 2, 2], [0, 0, 2, 1]], np.float32)
    assert O.nms(b, np.array([0.9, 0.8], np.float32), 0.5).tolist() == [0, 1]
    assert O.nms(b, np.array([0.9, 0.8], np.float32), 0.49).tolist() == [0]
    # ties in score: lower index first; empty input
    assert O.nms(boxes[[2, 2, 2]], np.array([0.5, 0.5, 0.5], np.float32), 0.5).tolist() == [0]
    assert O.nms(np.zeros((0, 4), np.float32), np.zeros(0, np.float32), 0.5).tolist() == []


def _random_boxes(rng, n, span=200.0):
    side = np.exp(rng.uniform(np.log(8), np.log(120), n))
    asp = np.exp(rng.uniform(np.log(0.5), np.log(2), n))
    w, h = side * np.sqrt(asp), side / np.sqrt(asp)
    cx, cy = rng.uniform(0, span, n), rng.uniform(0, span, n)
    return np.stack([cx - w / 2, cy - h / 2, cx + w / 2, cy + h / 2], 1).astype(np.float32)


def test_nms_matches_library_routine_and_invariants():
    rng = np.random.default_rng(3)
    for n, thr in ((50, 0.5), (300, 0.7), (400, 0.3)):
        boxes = _random_boxes(rng, n)
        scores = rng.permutation(n).astype(np.float32) / n          # distinct
        keep = O.nms(boxes, scores, thr)
        # kept boxes do not suppress each other; every dropped box is suppressed by a kept, higher-scored one
        for i, a in enumerate(keep):
            for b in keep[i + 1:]:
                assert not (O.iou(boxes[a], boxes[b]) > thr)
        kept = set(keep.tolist())
        for j in range(n):
            if j not in kept:
                assert any(scores[a] > scores[j] and O.iou(boxes[a], boxes[j]) > thr for a in keep)
        assert np.all(np.diff(scores[keep]) < 0)
        # idempotent, and invariant under a permutation of the input
        assert O.nms(boxes[keep], scores[keep], thr).tolist() == list(range(len(keep)))
        perm = rng.permutation(n)
        assert sorted(perm[O.nms(boxes[perm], scores[perm], thr)].tolist()) == sorted(keep.tolist())
    tv = pytest.importorskip("torchvision")
    import torch
    boxes = _random_boxes(rng, 500)
    scores = rng.permutation(500).astype(np.float32) / 500
    ref = tv.ops.nms(torch.from_numpy(boxes), torch.from_numpy(scores), 0.5).numpy()
    assert O.nms(boxes, scores, 0.5).tolist() == ref.tolist()


# ------------------------------------------------------------------------------------------ Soft-NMS
def test_soft_nms_worked_examples():
    boxes = np.array([[0, 0, 2, 2], [1, 0, 3, 2], [10, 10, 11, 11]], np.float32)   # IoU(0,1) = 2/6 = 1/3
    scores = np.array([0.9, 0.8, 0.5], np.float32)
    idx, sc = O.soft_nms(boxes, scores, 0.3, 0.5, 0.001, "linear")
    assert idx.tolist() == [0, 1, 2]
    assert np.allclose(sc, [0.9, 0.8 * (1 - 1 / 3), 0.5], rtol=1e-6)
    idx, sc = O.soft_nms(boxes, scores, 0.3, 0.5, 0.001, "gaussian")
    assert idx.tolist() == [0, 1, 2]
    assert np.allclose(sc, [0.9, 0.8 * math.exp(-(1 / 9) / 0.5), 0.5], rtol=1e-6)
    # below the IoU threshold the linear method leaves the score alone
    idx, sc = O.soft_nms(boxes, scores, 0.4, 0.5, 0.001, "linear")
    assert np.allclose(sc, [0.9, 0.8, 0.5])
    # the decayed score decides the order: 0.8 * (1 - 1/3) = 0.533 drops below an untouched 0.6
    idx, sc = O.soft_nms(boxes, np.array([0.9, 0.8, 0.6], np.float32), 0.3, 0.5, 0.001, "linear")
    assert idx.tolist() == [0, 2, 1]
    # min_score prunes
    idx, sc = O.soft_nms(boxes, scores, 0.3, 0.5, 0.52, "linear")
    assert idx.tolist() == [0, 1]


def test_soft_nms_without_overlap_is_a_score_sort():
    rng = np.random.default_rng(9)
    n = 40
    boxes = np.stack([np.arange(n) * 10.0, np.zeros(n), np.arange(n) * 10.0 + 5, np.full(n, 5.0)], 1).astype(np.float32)
    scores = rng.uniform(0.1, 1, n).astype(np.float32)
    for method in ("linear", "gaussian"):
        idx, sc = O.soft_nms(boxes, scores, 0.3, 0.5, 0.0, method)
        assert idx.tolist() == np.argsort(-scores, kind="stable").tolist()
        assert np.array_equal(sc, scores[idx])


# ------------------------------------------------------------------------------- deformable RoI pooling
# Pins of oracle/ops_ref.cpp deform_roi_pool_* (readings D1-D5).  The RoIAlign oracle it is
# compared with (oracle/raf_ref.cpp) is itself pinned in tests/test_oracle_forward.py / _backward.py.
from oracle import raf_ref as R  # noqa: E402


def _deform_case(seed=3, K=12, C=3, shapes=((1, 3, 40, 48), (1, 3, 20, 24)), P=(5, 6)):
    rng = np.random.default_rng(seed)
    feats = [rng.standard_normal(s) for s in shapes]
    scales = [0.25, 0.125]
    side = np.exp(rng.uniform(np.log(20), np.log(170), (K, 2)))
    cx, cy = rng.uniform(0, 190, K), rng.uniform(0, 160, K)
    rois = np.stack([np.zeros(K), cx - side[:, 0] / 2, cy - side[:, 1] / 2, cx + side[:, 0] / 2,
                     cy + side[:, 1] / 2], 1).astype(np.float32)
    off = rng.uniform(-0.6, 0.6, (K, 2) + P).astype(np.float32)
    return feats, scales, rois, off, P


def test_deform_zero_offset_is_roialign_bit_for_bit():
    feats, scales, rois, off, P = _deform_case()
    for g in (1, 2, 0):
        a = O.deform_roi_pool_forward(feats, scales, rois, None, 0.1, P, g)
        b = O.deform_roi_pool_forward(feats, scales, rois, np.zeros_like(off), 0.1, P, g)
        ref = R.forward(feats, scales, rois, P, g, True, 56.0, coord_f32=True)
        assert np.array_equal(a, ref) and np.array_equal(b, ref)
        a64 = O.deform_roi_pool_forward(feats, scales, rois, None, 0.1, P, g, f64=True)
        assert np.abs(a64 - R.forward(feats, scales, rois, P, g, True, 56.0, coord_f32=False)).max() < 1e-12


def test_deform_uniform_offset_is_a_translated_box():
    """offset (dx, dy) on EVERY bin moves all samples by gamma*(rw*dx, rh*dy) feature pixels = the RoI moved by
    that much divided by the level's scale in image pixels (f64 mode: exact up to rounding)."""
    feats, scales, rois, _, P = _deform_case(seed=4, K=8)
    gamma, dx, dy = 0.25, 0.3, -0.2
    off = np.zeros((len(rois), 2) + P, np.float32)
    off[:, 0], off[:, 1] = dx, dy
    got = O.deform_roi_pool_forward(feats, scales, rois, off, gamma, P, 2, f64=True)
    levels = R.assign_levels(rois, 2, 56.0)[0]
    moved = rois.astype(np.float64).copy()
    w, h = moved[:, 3] - moved[:, 1], moved[:, 4] - moved[:, 2]
    # feature-pixel shift gamma*rw*dx with rw = w*scale  ->  image-pixel shift gamma*w*dx (the scale cancels)
    sx, sy = gamma * w * np.float64(np.float32(dx)), gamma * h * np.float64(np.float32(dy))
    # the level map must see the ORIGINAL box: evaluate RoI by RoI on the level the original was assigned to
    for k in range(len(rois)):
        l = int(levels[k])
        r = np.array([[0, moved[k, 1] + sx[k], moved[k, 2] + sy[k], moved[k, 3] + sx[k], moved[k, 4] + sy[k]]])
        ref = _roialign_f64_single(feats[l], scales[l], r[0], P, 2)
        assert np.abs(got[k] - ref).max() < 1e-9


def _roialign_f64_single(feat, scale, roi, P, g):
    """Plain float64 RoIAlign of one box on one level, written out here (independent of both oracles)."""
    _, C, H, W = feat.shape
    PH, PW = P
    sx, sy = roi[1] * scale - 0.5, roi[2] * scale - 0.5
    bw, bh = (roi[3] * scale - 0.5 - sx) / PW, (roi[4] * scale - 0.5 - sy) / PH
    out = np.zeros((C, PH, PW))

    def axis(v, n):
        if v < -1 or v > n:
            return None
        v = max(v, 0.0)
        lo = int(v)
        if lo >= n - 1:
            return n - 1, n - 1, 1.0, 0.0
        return lo, lo + 1, 1 - (v - lo), v - lo
    for ph in range(PH):
        for pw in range(PW):
            for iy in range(g):
                ty = axis(sy + ph * bh + (iy + 0.5) * bh / g, H)
                if ty is None:
                    continue
                for ix in range(g):
                    tx = axis(sx + pw * bw + (ix + 0.5) * bw / g, W)
                    if tx is None:
                        continue
                    out[:, ph, pw] += (ty[2] * tx[2] * feat[0, :, ty[0], tx[0]] + ty[2] * tx[3] * feat[0, :, ty[0], tx[1]] +
                                       ty[3] * tx[2] * feat[0, :, ty[1], tx[0]] + ty[3] * tx[3] * feat[0, :, ty[1], tx[1]])
    return out / (g * g)


def test_deform_offset_of_one_bin_changes_that_bin_only_and_planes_are_x_then_y():
    feats, scales, rois, _, P = _deform_case(seed=5, K=4)
    base = O.deform_roi_pool_forward(feats, scales, rois, None, 0.2, P, 2)
    off = np.zeros((4, 2) + P, np.float32)
    off[1, 0, 2, 3] = 0.5
    got = O.deform_roi_pool_forward(feats, scales, rois, off, 0.2, P, 2)
    diff = got != base
    assert diff[1, :, 2, 3].any()
    diff[1, :, 2, 3] = False
    assert not diff.any()
    # x-ramp feature: an x offset moves the value by gamma*rw*dx*slope, a y offset leaves it unchanged
    H, W = 40, 48
    ramp = np.broadcast_to(np.arange(W, dtype=np.float64)[None, None, None, :] * 2.0, (1, 1, H, W)).copy()
    roi = np.array([[0, 40, 40, 120, 100]], np.float32)     # level 0 at scale 0.25: 20 x 15 px, interior
    P2 = (3, 4)
    z = O.deform_roi_pool_forward([ramp], [0.25], roi, None, 0.1, P2, 2, f64=True)
    ox = np.zeros((1, 2) + P2, np.float32); ox[0, 0] = 0.25
    oy = np.zeros((1, 2) + P2, np.float32); oy[0, 1] = 0.25
    rw = (120 - 40) * 0.25
    g32 = np.float64(np.float32(0.1))      # gamma is a float32 argument
    assert np.abs(O.deform_roi_pool_forward([ramp], [0.25], roi, ox, 0.1, P2, 2, f64=True) - (z + g32 * rw * 0.25 * 2.0)).max() < 1e-9
    assert np.abs(O.deform_roi_pool_forward([ramp], [0.25], roi, oy, 0.1, P2, 2, f64=True) - z).max() < 1e-12


def test_deform_backward_adjoint_and_finite_differences():
    feats, scales, rois, off, P = _deform_case(seed=6, K=6)
    gamma = 0.15
    rng = np.random.default_rng(7)
    gout = rng.standard_normal((len(rois), feats[0].shape[1]) + P)
    out = O.deform_roi_pool_forward(feats, scales, rois, off, gamma, P, 2, f64=True)
    gf, goff = O.deform_roi_pool_backward(feats, scales, gout, rois, off, gamma, 2, f64=True)
    # feature gradient = transpose of the (linear in F) forward:  <A x, g> = <x, A^T g>
    lhs = float((out * gout).sum())
    rhs = float(sum((f * g).sum() for f, g in zip(feats, gf)))
    assert abs(lhs - rhs) < 1e-10 * max(1.0, abs(lhs))
    # offset gradient = derivative of the forward: central differences on a few entries (f64 forward; an entry is
    # skipped when a sample sits within the step of a pixel boundary, where the forward has a kink)
    eps, checked = 1e-4, 0
    for (k, a, ph, pw) in [(0, 0, 1, 2), (1, 1, 0, 0), (2, 0, 4, 5), (3, 1, 2, 2), (4, 0, 3, 1), (5, 1, 1, 4)]:
        op, om = off.astype(np.float64).copy(), off.astype(np.float64).copy()
        # float32 offsets: perturb by a float32-exact amount
        d = np.float32(off[k, a, ph, pw] + eps) - off[k, a, ph, pw]
        op[k, a, ph, pw] += d; om[k, a, ph, pw] -= d
        fp = O.deform_roi_pool_forward(feats, scales, rois, op.astype(np.float32), gamma, P, 2, f64=True)
        fm = O.deform_roi_pool_forward(feats, scales, rois, om.astype(np.float32), gamma, P, 2, f64=True)
        dp = np.float64(np.float32(op[k, a, ph, pw])) - np.float64(off[k, a, ph, pw])
        dm = np.float64(off[k, a, ph, pw]) - np.float64(np.float32(om[k, a, ph, pw]))
        num = float(((fp - fm) * gout).sum()) / (dp + dm)
        # second difference small <=> no kink inside the step
        curv = float((np.abs(fp - 2 * out + fm) * np.abs(gout)).sum())
        if curv > 1e-9:
            continue
        assert abs(num - goff[k, a, ph, pw]) < 1e-6 * max(1.0, abs(num))
        checked += 1
    assert checked >= 3
    # constant map: the forward does not depend on the offsets (inside the map)
    const = [np.full(f.shape, 2.5) for f in feats]
    inner = rois.copy(); inner[:, 1:] = [60, 50, 110, 95]
    _, g0 = O.deform_roi_pool_backward(const, scales, gout, inner, off * 0.1, gamma, 2, f64=True)
    assert np.abs(g0).max() < 1e-12
    # spec mode (fp32 coordinates) stays within coordinate rounding of the f64 mode
    gf32, goff32 = O.deform_roi_pool_backward(feats, scales, gout, rois, off, gamma, 2, f64=False)
    assert max(np.abs(a - b).max() for a, b in zip(gf, gf32)) < 1e-3


# --------------------------------------------------------------------------- RoIAlign -> first FC (fused op)
def test_roi_align_fc_oracle_flatten_order_rounding_and_linearity():
    """Pins of O.roi_align_fc_forward (readings F1-F3): a selection matrix returns single rounded RoI features in
    (ph, pw, c) order; the product is linear in the weight and adds the bias; a loop restatement on a tiny case."""
    rng = np.random.default_rng(9)
    feats = [rng.standard_normal((1, 8, 24, 30)), rng.standard_normal((1, 8, 12, 15))]
    scales = [0.25, 0.125]
    rois = np.array([[0, 10, 12, 70, 60], [0, 5, 5, 110, 90], [0, 30, 20, 50, 44]], np.float32)
    P = (3, 4)
    x = R.forward(feats, scales, rois, P, 2, True, 56.0, coord_f32=True)
    Kd = P[0] * P[1] * 8
    # selection: output n picks flattened index sel[n]
    sel = np.array([0, 7, 8, 8 * 4 + 3, Kd - 1])
    W = np.zeros((len(sel), Kd)); W[np.arange(len(sel)), sel] = 1.0
    got = O.roi_align_fc_forward(feats, scales, rois, W, None, P, 2, True, dtype="bf16")
    for n, s in enumerate(sel):
        ph, pw, c = s // (P[1] * 8), (s // 8) % P[1], s % 8
        want = x[:, c, ph, pw]
        # bf16 keeps an 8-bit significand, round to nearest even (np.round rounds halves to even); the value is first
        # rounded to fp32, which cannot move an 8-bit rounding decision except at exact ties (none in random data)
        m, e = np.frexp(want)
        q = np.ldexp(np.round(m * 256.0) / 256.0, e)
        assert np.array_equal(got[:, n], q)
    # f32 "rounding" keeps the features; linearity and bias
    W1, W2 = rng.standard_normal((6, Kd)), rng.standard_normal((6, Kd))
    b = rng.standard_normal(6)
    f = lambda w, bb: O.roi_align_fc_forward(feats, scales, rois, w, bb, P, 2, True, dtype="f32")
    assert np.abs(f(2 * W1 - W2, b) - (2 * f(W1, None) - f(W2, None) + b)).max() < 1e-9
    # loop restatement
    xr = x.astype(np.float32).astype(np.float64)
    want = np.zeros((3, 6))
    for k in range(3):
        for n in range(6):
            acc = 0.0
            for ph in range(P[0]):
                for pw in range(P[1]):
                    for c in range(8):
                        acc += xr[k, c, ph, pw] * W1[n, (ph * P[1] + pw) * 8 + c]
            want[k, n] = acc
    assert np.abs(f(W1, None) - want).max() < 1e-10
