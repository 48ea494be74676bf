"""Pins for the oracle's backward: the forward operator A is linear and pinned
by test_oracle_forward.py, so its transpose is pinned by (i) the adjoint identity <Ax,g> = <x,A^T g>,
(ii) an explicit dense A assembled by forwarding unit impulses, (iii) an independent library's
autograd, (iv) the worked example of config 1, plus hand-computed cases and mode semantics.
"""
import os

import numpy as np
import pytest

from conftest import read_golden
from oracle import raf_ref as R
from paper_1906_07155_b200 import inputs


def test_adjoint_identity_config1_f64():
    wl = inputs.make_workload(1)
    out = R.forward(wl.feats, [1.0], wl.rois, (7, 7), 2, True, coord_f32=False)
    g, S = R.backward([(1, 4, 16, 16)], [1.0], wl.grad_out, wl.rois, (7, 7), 2, True, coord_f32=False)
    lhs = float((out * wl.grad_out.astype(np.float64)).sum())
    rhs = float((g[0] * wl.feats[0].astype(np.float64)).sum())
    assert abs(lhs - rhs) < 1e-12 * max(1.0, abs(lhs))


@pytest.mark.parametrize("f32", [False, True])
@pytest.mark.parametrize("g,aligned,P", [(2, True, (7, 7)), (0, False, (5, 3)), (3, True, (2, 6)), (1, False, (7, 7))])
def test_adjoint_identity_pyramid(f32, g, aligned, P):
    # multi-level, boxes partly outside the image, two images
    wl = inputs.make_workload(5, n_img=2, per_img=20, channels=3)
    cfg = wl.cfg
    rng = np.random.default_rng(9)
    gout = rng.standard_normal((cfg.K, 3, *P))
    out = R.forward(wl.feats, cfg.scales, wl.rois, P, g, aligned, coord_f32=f32)
    grads, S = R.backward(cfg.level_shapes, cfg.scales, gout, wl.rois, P, g, aligned, coord_f32=f32)
    lhs = float((out * gout).sum())
    rhs = sum(float((gr * f.astype(np.float64)).sum()) for gr, f in zip(grads, wl.feats))
    assert abs(lhs - rhs) < 1e-11 * max(1.0, abs(lhs))
    # S bounds |grad| element-wise and is zero exactly where nothing was scattered
    for gr, s in zip(grads, S):
        assert np.all(np.abs(gr) <= s + 1e-15)
        assert np.all((s == 0) <= (gr == 0))


def test_dense_operator_brute_force_config1():
    """Build A (K*C*PH*PW x N*C*H*W) column by column from unit impulses; compare A^T g."""
    wl = inputs.make_workload(1)
    C, H, W = 4, 16, 16
    K, PH, PW = 8, 7, 7
    # channels are independent and identical: assemble A for one channel
    A = np.zeros((K * PH * PW, H * W))
    for j in range(H * W):
        e = np.zeros((1, 1, H, W))
        e.reshape(-1)[j] = 1.0
        A[:, j] = R.forward([e], [1.0], wl.rois, (PH, PW), 2, True, coord_f32=True).reshape(-1)
    grads, _ = R.backward([(1, C, H, W)], [1.0], wl.grad_out, wl.rois, (PH, PW), 2, True, coord_f32=True)
    for c in range(C):
        gc = wl.grad_out[:, c].astype(np.float64).reshape(-1)
        assert np.allclose(A.T @ gc, grads[0][0, c].reshape(-1), atol=1e-12)


def test_hand_computed_identity_crop_transpose():
    # scale 1, aligned, RoI (0,0,7,7), g=1: forward is the crop F[0:7,0:7] -> backward pastes gout
    rng = np.random.default_rng(1)
    gout = rng.standard_normal((1, 1, 7, 7))
    g, S = R.backward([(1, 1, 16, 16)], [1.0], gout, [[0, 0, 0, 7, 7]], (7, 7), 1, True, coord_f32=False)
    exp = np.zeros((16, 16)); exp[:7, :7] = gout[0, 0]
    assert np.allclose(g[0][0, 0], exp, atol=1e-15)
    assert np.allclose(S[0][0, 0], np.abs(exp), atol=1e-15)
    # 2x2 block mean (RoI .5..7.5): each gout value spreads 1/4 to its 2x2 block
    g, _ = R.backward([(1, 1, 16, 16)], [1.0], gout, [[0, .5, .5, 7.5, 7.5]], (7, 7), 2, True, coord_f32=False)
    exp = np.zeros((16, 16))
    for i in range(7):
        for j in range(7):
            exp[i:i + 2, j:j + 2] += 0.25 * gout[0, 0, i, j]
    assert np.allclose(g[0][0, 0], exp, atol=1e-15)


def test_outside_samples_give_no_gradient_and_count_is_full():
    # constant-map pin transposed: RoI (-4,2,3,9) -> columns with valid fraction [0,0,0,.5,1,1,1];
    # total scattered mass = sum_bins gout * fraction
    gout = np.ones((1, 1, 7, 7))
    g, _ = R.backward([(1, 1, 16, 16)], [1.0], gout, [[0, -4, 2, 3, 9]], (7, 7), 2, True, coord_f32=False)
    assert np.isclose(g[0].sum(), 7 * (0.5 + 3), atol=1e-13)
    assert np.all(g[0][0, 0, :, 4:] == 0)


def test_overwrite_vs_accumulate_and_invalid_batch():
    wl = inputs.make_workload(1)
    base = [np.full((1, 4, 16, 16), 2.0)]
    g0, _ = R.backward([(1, 4, 16, 16)], [1.0], wl.grad_out, wl.rois, (7, 7), 2, True)
    g1, _ = R.backward([(1, 4, 16, 16)], [1.0], wl.grad_out, wl.rois, (7, 7), 2, True, accumulate_into=base)
    assert np.allclose(g1[0], g0[0] + 2.0, atol=1e-14)
    rois = wl.rois.copy(); rois[:, 0] = 3
    gz, S = R.backward([(1, 4, 16, 16)], [1.0], wl.grad_out, rois, (7, 7), 2, True)
    assert np.all(gz[0] == 0) and np.all(S[0] == 0)


def test_worked_example_config1(golden_dir):
    gd = read_golden(os.path.join(golden_dir, "config1_f64.txt"))
    wl = inputs.make_workload(1)
    if not np.allclose(wl.rois[0], gd["roi0"], atol=1e-5):
        pytest.skip("numpy stream differs from the one the golden values were drawn with")
    assert np.allclose(wl.grad_out[0, 0, 0, :3], gd["gout_0_0_0_0to2"], atol=1e-7)
    g, _ = R.backward([(1, 4, 16, 16)], [1.0], wl.grad_out, wl.rois, (7, 7), 2, True, coord_f32=False)
    g = g[0]
    assert abs(g.sum() - gd["sum_grad"]) < 1e-7
    assert abs(np.abs(g).sum() - gd["sum_abs_grad"]) < 1e-7
    assert abs(g[0, 0, 8, 8] - gd["grad_0_0_8_8"]) < 1e-8
    assert abs(g[0, 2, 3, 11] - gd["grad_0_2_3_11"]) < 1e-8
    assert int((g != 0).sum()) == int(gd["grad_nonzero"])
    out = R.forward(wl.feats, [1.0], wl.rois, (7, 7), 2, True, coord_f32=False)
    assert abs((out * wl.grad_out).sum() - gd["inner_product"]) < 1e-9


def test_against_independent_library_autograd():
    tv = pytest.importorskip("torchvision")
    import torch
    rng = np.random.default_rng(13)
    for aligned, g, scale, P in [(True, 2, 0.25, (7, 7)), (False, 2, 0.5, (3, 5)), (True, 0, 1.0, (4, 4)),
                                 (False, 3, 0.25, (14, 14)), (True, 1, 0.5, (7, 2))]:
        F = torch.from_numpy(rng.standard_normal((2, 3, 18, 22))).requires_grad_(True)
        K = 9
        xs = np.sort(rng.uniform(-0.2 * 22 / scale, 1.2 * 22 / scale, (K, 2)), axis=1)
        ys = np.sort(rng.uniform(-0.2 * 18 / scale, 1.2 * 18 / scale, (K, 2)), axis=1)
        rois = np.stack([rng.integers(0, 2, K), xs[:, 0], ys[:, 0], xs[:, 1], ys[:, 1]], 1).astype(np.float32)
        gout = rng.standard_normal((K, 3, *P))
        o = tv.ops.roi_align(F, torch.from_numpy(rois.astype(np.float64)), P, scale, g, aligned)
        o.backward(torch.from_numpy(gout))
        got, _ = R.backward([(2, 3, 18, 22)], [scale], gout, rois, P, g, aligned, coord_f32=False)
        assert np.allclose(got[0], F.grad.numpy(), atol=1e-10), (aligned, g, scale, P)


def test_footprint_union_matches_survey_and_backward_support(golden_dir):
    gd = read_golden(os.path.join(golden_dir, "level_histograms.txt"))
    for i in (2, 4):
        wl = inputs.make_workload(i, with_feats=False, with_grad=False)
        cfg = wl.cfg
        shapes = [(s[0], 1, s[2], s[3]) for s in cfg.level_shapes]
        masks = R.footprint(shapes, cfg.scales, wl.rois, cfg.out_size, 2, True)
        assert sum(int(m.sum()) for m in masks) == int(gd[f"union{i}"])
    # the footprint is exactly the support of S from the backward
    wl = inputs.make_workload(2, n_img=2, per_img=16, channels=1)
    cfg = wl.cfg
    masks = R.footprint(cfg.level_shapes, cfg.scales, wl.rois, (7, 7), 2, True)
    _, S = R.backward(cfg.level_shapes, cfg.scales, np.ones((cfg.K, 1, 7, 7)), wl.rois, (7, 7), 2, True)
    for m, s in zip(masks, S):
        # weights can be exactly 0 at integer coordinates: support(S) is a subset of the footprint
        assert np.all((s[:, 0] > 0) <= (m > 0))
        assert (s[:, 0] > 0).sum() >= 0.9 * m.sum()
