"""Pins for the oracle's forward (readings S5-S8): closed forms, hand-computed
integer-aligned cases, the edge rule, invariants, an independent library routine, and the worked
example of config 1.  Chosen so that a dropped term, wrong sign/index or transposed operand fails.
"""
import os

import numpy as np
import pytest

from conftest import read_golden
from oracle import raf_ref as R
from paper_1906_07155_b200 import inputs


def fwd1(feat2d_or_4d, rois, scale=1.0, P=7, g=2, aligned=True, f32=False):
    f = np.asarray(feat2d_or_4d, np.float64)
    if f.ndim == 2:
        f = f[None, None]
    rois = np.asarray(rois, np.float32).reshape(-1, 5)
    P = P if isinstance(P, tuple) else (P, P)
    return R.forward([f], [scale], rois, P, g, aligned, coord_f32=f32)


RNG = np.random.default_rng(0)
F16 = RNG.standard_normal((16, 16))


@pytest.mark.parametrize("f32", [False, True])
def test_constant_map_inside_is_constant(f32):
    out = fwd1(np.full((16, 16), 3.0), [0, 1.3, 2.1, 11.9, 12.7], f32=f32)
    assert np.allclose(out, 3.0, atol=1e-6 if f32 else 1e-14)


def test_constant_map_partially_outside_counts_all_samples():
    # SURVEY pin: 16x16 map == 3, RoI (-4,2,3,9), 7x7, g=2, aligned -> columns 3*[0,0,0,.5,1,1,1]
    out = fwd1(np.full((16, 16), 3.0), [0, -4, 2, 3, 9])[0, 0]
    assert np.allclose(out, 3.0 * np.tile([0, 0, 0, 0.5, 1, 1, 1], (7, 1)), atol=1e-14)
    # same box rotated onto the y axis -> rows (catches x/y swap)
    out = fwd1(np.full((16, 16), 3.0), [0, 2, -4, 9, 3])[0, 0]
    assert np.allclose(out, 3.0 * np.tile([0, 0, 0, 0.5, 1, 1, 1], (7, 1)).T, atol=1e-14)


@pytest.mark.parametrize("P,g", [((7, 7), 2), ((7, 7), 3), ((5, 9), 2), ((14, 14), 1)])
def test_affine_map_gives_bin_centre_value(P, g):
    yy, xx = np.mgrid[0:32, 0:40]
    a, b, d = 2.0, -3.0, 5.0
    ramp = a * xx + b * yy + d
    roi = tuple(float(np.float32(v)) for v in (2.3, 4.1, 30.9, 25.7))   # boxes are fp32 at the ABI
    scale = 0.5
    out = fwd1(ramp, [0, *roi], scale=scale, P=P, g=g)[0, 0]
    sx, sy = roi[0] * scale - 0.5, roi[1] * scale - 0.5
    bw, bh = (roi[2] - roi[0]) * scale / P[1], (roi[3] - roi[1]) * scale / P[0]
    exp = np.array([[a * (sx + (pw + .5) * bw) + b * (sy + (ph + .5) * bh) + d
                     for pw in range(P[1])] for ph in range(P[0])])
    assert np.allclose(out, exp, atol=1e-11)


def test_integer_aligned_identity_crop():
    out = fwd1(F16, [0, 0, 0, 7, 7], g=1)[0, 0]
    assert np.allclose(out, F16[:7, :7], atol=1e-15)
    # non-square crop: catches H/W and PH/PW transposition
    out = fwd1(F16, [0, 2, 1, 7, 10], P=(9, 5), g=1)[0, 0]
    assert np.allclose(out, F16[1:10, 2:7], atol=1e-15)


def test_integer_aligned_stencil_g2():
    k = np.zeros((7, 16))
    k[0, 0], k[0, 1] = 0.875, 0.125          # -0.25 clamps to 0
    for p in range(1, 7):
        k[p, p - 1], k[p, p], k[p, p + 1] = .125, .75, .125
    out = fwd1(F16, [0, 0, 0, 7, 7], g=2)[0, 0]
    assert np.allclose(out, k @ F16 @ k.T, atol=1e-14)


def test_half_pixel_box_is_2x2_block_mean():
    blk = 0.25 * (F16[:7, :7] + F16[1:8, :7] + F16[:7, 1:8] + F16[1:8, 1:8])
    for g in (1, 2):
        assert np.allclose(fwd1(F16, [0, .5, .5, 7.5, 7.5], g=g)[0, 0], blk, atol=1e-14)
        assert np.allclose(fwd1(F16, [0, 2, 2, 30, 30], scale=0.25, g=g)[0, 0], blk, atol=1e-14)
        # aligned=False: no half-pixel shift (reading S5)
        assert np.allclose(fwd1(F16, [0, 0, 0, 7, 7], g=g, aligned=False)[0, 0], blk, atol=1e-14)


def test_not_aligned_clamps_roi_size_to_one():
    # aligned=False: rw, rh >= 1 -> a zero-size box at (3,4) samples inside [3,4]x[4,5]:
    # P=1,g=1 -> sample at (4.5, 3.5) = mean of the 2x2 block at row 4, col 3
    out = fwd1(F16, [0, 3, 4, 3, 4], P=1, g=1, aligned=False)[0, 0, 0, 0]
    assert np.isclose(out, 0.25 * (F16[4, 3] + F16[4, 4] + F16[5, 3] + F16[5, 4]), atol=1e-15)
    # aligned=True: no clamp -> all samples coincide at (3.5, 2.5)
    out = fwd1(F16, [0, 3, 4, 3, 4], P=1, g=2, aligned=True)[0, 0, 0, 0]
    assert np.isclose(out, 0.25 * (F16[3, 2] + F16[3, 3] + F16[4, 2] + F16[4, 3]), atol=1e-15)


def test_edge_rule():
    # P=1, g=1, aligned: the single sample sits at the box centre minus 0.5
    ramp = np.tile(np.arange(16.0), (16, 1))

    def at(x, y=3.0, m=ramp):
        return fwd1(m, [0, x + 0.5 - 1, y + 0.5 - 1, x + 0.5 + 1, y + 0.5 + 1], P=1, g=1)[0, 0, 0, 0]
    assert at(15.5) == 15.0            # clamps to the edge pixel
    assert at(16.0) == 15.0            # closed band [-1, W]
    assert at(16.0001) == 0.0          # outside: contributes 0
    assert at(-1.0, m=ramp + 7) == 7.0
    assert at(-1.0001, m=ramp + 7) == 0.0
    assert at(7.25) == 7.25
    col = ramp.T
    assert at(3.0, 16.0, col) == 15.0 and at(3.0, 16.0001, col) == 0.0
    assert at(3.0, -1.0, col + 7) == 7.0 and at(3.0, -1.0001, col + 7) == 0.0


def test_adaptive_sampling_ratio():
    # sampling_ratio = 0: gh = ceil(rh/PH), gw = ceil(rw/PW) (reading S7)
    roi = [0, 1, 2, 15, 9]     # rw=14 -> bw=2 -> gw=2 ; rh=7 -> bh=1 -> gh=1
    assert np.allclose(fwd1(F16, roi, g=0), _manual(F16, roi, 7, 7, 1, 2), atol=1e-14)
    roi = [0, 1, 1, 15.5, 12]  # bw = 14.5/7 -> gw=3 ; bh = 11/7 -> gh=2
    assert np.allclose(fwd1(F16, roi, g=0), _manual(F16, roi, 7, 7, 2, 3), atol=1e-14)
    # aligned + non-positive extent: empty loops, output 0
    assert np.all(fwd1(F16, [0, 9, 9, 3, 3], g=0) == 0)


def _manual(F, roi, PH, PW, gh, gw):
    """Brute force with explicit grids; bilinear through np.interp along each axis (interior only)."""
    sx, sy = roi[1] - .5, roi[2] - .5
    bw, bh = (roi[3] - roi[1]) / PW, (roi[4] - roi[2]) / PH
    out = np.zeros((PH, PW))
    H, W = F.shape
    for ph in range(PH):
        for pw in range(PW):
            acc = 0.0
            for iy in range(gh):
                y = min(max(sy + ph * bh + (iy + .5) * bh / gh, 0), H - 1)
                rowvals = np.array([np.interp(y, np.arange(H), F[:, c]) for c in range(W)])
                for ix in range(gw):
                    x = min(max(sx + pw * bw + (ix + .5) * bw / gw, 0), W - 1)
                    acc += np.interp(x, np.arange(W), rowvals)
            out[ph, pw] = acc / (gh * gw)
    return out


def test_matches_interp_brute_force_random_boxes():
    rng = np.random.default_rng(3)
    F = rng.standard_normal((20, 24))
    for _ in range(10):
        x = np.sort(rng.uniform(0, 24, 2)); y = np.sort(rng.uniform(0, 20, 2))
        roi = [float(np.float32(v)) for v in (0, x[0], y[0], x[1], y[1])]   # fp32 at the ABI
        got = fwd1(F, roi, P=(5, 6), g=2)[0, 0]
        assert np.allclose(got, _manual(F, roi, 5, 6, 2, 2), atol=1e-12)


def test_invariants_channel_perm_translation_transpose_routing():
    rng = np.random.default_rng(5)
    wl = inputs.make_workload(2, n_img=2, per_img=24, channels=3)
    cfg = wl.cfg
    out = R.forward(wl.feats, cfg.scales, wl.rois, (7, 7), 2, True, coord_f32=False)
    # channel independence
    one = R.forward([f[:, 1:2] for f in wl.feats], cfg.scales, wl.rois, (7, 7), 2, True, coord_f32=False)
    assert np.array_equal(out[:, 1:2], one)
    # RoI permutation
    p = rng.permutation(cfg.K)
    assert np.array_equal(R.forward(wl.feats, cfg.scales, wl.rois[p], (7, 7), 2, True, coord_f32=False), out[p])
    # level routing (C5): row k equals single-level forward on level_k with that level's scale
    levels = R.assign_levels(wl.rois, 4, 56.0)[0]
    assert len(set(levels.tolist())) == 4
    for k in range(0, cfg.K, 5):
        l = levels[k]
        single = R.forward([wl.feats[l]], [cfg.scales[l]], wl.rois[k:k + 1], (7, 7), 2, True, coord_f32=False)
        assert np.array_equal(single[0], out[k])
    # batch routing: image 1's RoIs do not see image 0
    f2 = [f.copy() for f in wl.feats]
    for f in f2:
        f[0] = 0
    o2 = R.forward(f2, cfg.scales, wl.rois, (7, 7), 2, True, coord_f32=False)
    assert np.all(o2[:24] == 0) and np.array_equal(o2[24:], out[24:])
    # x/y transpose
    ft = [np.ascontiguousarray(f.transpose(0, 1, 3, 2)) for f in wl.feats]
    rt = wl.rois[:, [0, 2, 1, 4, 3]]
    ot = R.forward(ft, cfg.scales, rt, (7, 7), 2, True, coord_f32=False)
    assert np.allclose(ot, out.transpose(0, 1, 3, 2), atol=1e-13)
    # integer-pixel translation of map + RoI (interior boxes, single level, stride 1)
    F = rng.standard_normal((1, 2, 40, 40))
    roi = np.array([[0, 5.2, 6.1, 17.7, 19.3]], np.float32)
    a = R.forward([F], [1.0], roi, (7, 7), 2, True, coord_f32=False)
    Fs = np.roll(F, (3, 4), axis=(2, 3))
    b = R.forward([Fs], [1.0], roi + np.float32([0, 4, 3, 4, 3]), (7, 7), 2, True, coord_f32=False)
    assert np.allclose(a, b, atol=1e-5)   # fp32 box corners shift by exact integers only approximately


def test_invalid_batch_index_gives_zero_row():
    rois = [[-1, 1, 1, 9, 9], [1, 1, 1, 9, 9], [0.5, 1, 1, 9, 9], [np.nan, 1, 1, 9, 9], [0, 1, 1, 9, 9]]
    out = fwd1(F16, rois)
    assert np.all(out[:4] == 0) and np.any(out[4] != 0)


def test_spec_mode_close_to_f64_mode():
    wl = inputs.make_workload(1)
    a = R.forward(wl.feats, [1.0], wl.rois, (7, 7), 2, True, coord_f32=True)
    b = R.forward(wl.feats, [1.0], wl.rois, (7, 7), 2, True, coord_f32=False)
    assert 0 < np.abs(a - b).max() < 2e-5


def test_worked_example_config1(golden_dir):
    g = read_golden(os.path.join(golden_dir, "config1_f64.txt"))
    wl = inputs.make_workload(1)
    if not np.allclose(wl.rois[0], g["roi0"], atol=1e-5):
        pytest.skip("numpy stream differs from the one the golden values were drawn with")
    assert np.allclose(wl.feats[0][0, 0, 0, :3], g["feat_0_0_0_0to2"], atol=1e-7)
    out = R.forward(wl.feats, [1.0], wl.rois, (7, 7), 2, True, coord_f32=False)
    assert abs(out.sum() - g["sum_out"]) < 1e-7
    assert abs(np.abs(out).sum() - g["sum_abs_out"]) < 1e-7
    assert abs(out[0, 0, 0, 0] - g["out_0_0_0_0"]) < 1e-8
    assert abs(out[3, 1, 2, 5] - g["out_3_1_2_5"]) < 1e-8
    assert abs(out[7, 3, 6, 6] - g["out_7_3_6_6"]) < 1e-8


def test_against_independent_library_routine():
    tv = pytest.importorskip("torchvision")
    import torch
    rng = np.random.default_rng(11)
    F = rng.standard_normal((2, 3, 18, 22))
    Ft = torch.from_numpy(F)
    n = 0
    for aligned in (True, False):
        for g in (0, 1, 2, 3):
            for scale in (1.0, 0.5, 0.25):
                for P in ((3, 3), (7, 7), (14, 5)):
                    K = 6
                    W_img, H_img = 22 / scale, 18 / scale
                    xs = rng.uniform(-0.3 * W_img, 1.3 * W_img, (K, 2))
                    ys = rng.uniform(-0.3 * H_img, 1.3 * H_img, (K, 2))
                    kind = rng.integers(0, 4, K)
                    for k in range(K):
                        if kind[k] == 0:    # normal
                            xs[k].sort(); ys[k].sort()
                        elif kind[k] == 1:  # zero width
                            xs[k, 1] = xs[k, 0]; ys[k].sort()
                        elif kind[k] == 2:  # x reversed
                            xs[k] = np.sort(xs[k])[::-1]; ys[k].sort()
                        else:               # both reversed
                            xs[k] = np.sort(xs[k])[::-1]; ys[k] = np.sort(ys[k])[::-1]
                    if g == 0 and aligned:
                        # reading S7: the library raises on adaptive+aligned+negative extent
                        xs.sort(axis=1); ys.sort(axis=1)
                    rois = np.stack([rng.integers(0, 2, K), xs[:, 0], ys[:, 0], xs[:, 1], ys[:, 1]], 1).astype(np.float32)
                    ref = tv.ops.roi_align(Ft, torch.from_numpy(rois.astype(np.float64)), P, scale, g, aligned).numpy()
                    got = R.forward([F], [scale], rois, P, g, aligned, coord_f32=False)
                    assert np.allclose(got, ref, atol=1e-10), (aligned, g, scale, P)
                    n += K
    assert n >= 400
