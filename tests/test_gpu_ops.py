"""GPU parity of the SURVEY 8(f) operations (RoIPool-max, NMS, Soft-NMS) against oracle/ops_ref.cpp, through the
C ABI binding.  Index / selection results are bit-exact; RoIPool values are copies of inputs (bit-exact)."""
import numpy as np
import pytest
import torch

from oracle import ops_ref as O
from paper_1906_07155_b200 import binding as B
from paper_1906_07155_b200 import inputs
import raf_testlib as T

pytestmark = pytest.mark.gpu


def _pool_case(wl, dtype, layout):
    cfg = wl.cfg
    PH, PW = cfg.out_size
    K, C = cfg.K, cfg.channels
    feats, exact = T.device_feats(wl.feats, dtype, layout)
    rois = torch.from_numpy(wl.rois).cuda()
    out = T.empty_layout((K, C, PH, PW), feats[0].dtype, layout, fill=float("nan"))
    arg = torch.full_like(out, -7, dtype=torch.int32)
    assert arg.stride() == out.stride()
    B.roi_pool_fpn_forward(feats, cfg.scales, rois, out, arg, cfg.finest_scale)
    torch.cuda.synchronize()
    ref, aref = O.roi_pool_forward(exact, cfg.scales, wl.rois, (PH, PW), cfg.finest_scale)
    assert np.array_equal(arg.cpu().numpy(), aref)
    assert np.array_equal(out.to(torch.float64).cpu().numpy(), ref)
    return feats, rois, arg, aref


@pytest.mark.parametrize("layout", ["cl", "nchw"])
@pytest.mark.parametrize("index,dtype,kw", [
    (1, "f32", {}),
    (2, "f32", dict(n_img=2, per_img=150, channels=32)),
    (3, "f16", dict(n_img=1, per_img=200, channels=40)),
    (4, "bf16", dict(n_img=2, per_img=40, channels=24)),
    (5, "bf16", dict(n_img=3, per_img=100, channels=16)),
])
def test_roi_pool_forward_backward(index, dtype, kw, layout):
    wl = inputs.make_workload(index, **kw)
    cfg = wl.cfg
    feats, rois, arg, aref = _pool_case(wl, dtype, layout)
    go_t = torch.from_numpy(wl.grad_out).to(T.TORCH_DTYPE[dtype])
    go = T.to_layout(go_t.cuda(), layout)
    grads = [T.empty_layout(s, torch.float32, layout, fill=float("nan")) for s in cfg.level_shapes]
    B.roi_pool_fpn_backward(grads, cfg.scales, go, arg, rois, cfg.finest_scale)
    torch.cuda.synchronize()
    ge = go_t.to(torch.float64).numpy()
    ref = O.roi_pool_backward(cfg.level_shapes, cfg.scales, ge, aref, wl.rois, cfg.finest_scale)
    S = O.roi_pool_backward(cfg.level_shapes, cfg.scales, np.abs(ge), aref, wl.rois, cfg.finest_scale)
    T.assert_backward_close([g.to(torch.float64).cpu().numpy() for g in grads], ref, S)
    # accumulate mode adds onto the existing contents
    B.roi_pool_fpn_backward(grads, cfg.scales, go, arg, rois, cfg.finest_scale, B.RAF_ACCUMULATE)
    torch.cuda.synchronize()
    T.assert_backward_close([g.to(torch.float64).cpu().numpy() for g in grads], [2 * r for r in ref], [2 * s for s in S])


def test_roi_pool_degenerate_rois_and_no_argmax():
    wl = inputs.make_workload(2, n_img=2, per_img=16, channels=8)
    cfg = wl.cfg
    r = wl.rois.copy()
    r[0, 0] = 5.0                 # invalid batch index
    r[1, 1:] = [10, 10, 10, 10]   # zero extent: one pixel
    r[2, 1:] = [30, 40, 20, 10]   # reversed
    r[3, 1:] = [-500, -500, -400, -400]   # wholly outside
    r[4, 1:] = [1300, 700, 3000, 3000]    # partly outside
    wl.rois[:] = r
    _pool_case(wl, "f32", "cl")
    feats, exact = T.device_feats(wl.feats, "f32", "cl")
    out = T.empty_layout((cfg.K, cfg.channels, 7, 7), torch.float32, "cl", fill=float("nan"))
    B.roi_pool_fpn_forward(feats, cfg.scales, torch.from_numpy(wl.rois).cuda(), out, None, cfg.finest_scale)
    torch.cuda.synchronize()
    assert np.array_equal(out.double().cpu().numpy(), O.roi_pool_forward(exact, cfg.scales, wl.rois, (7, 7), cfg.finest_scale)[0])


def _boxes(rng, n, span):
    side = np.exp(rng.uniform(np.log(8), np.log(300), n))
    asp = np.exp(rng.uniform(np.log(0.5), np.log(2), n))
    w, h = side * np.sqrt(asp), side / np.sqrt(asp)
    cx, cy = rng.uniform(0, span, n), rng.uniform(0, span * 0.6, n)
    return np.stack([cx - w / 2, cy - h / 2, cx + w / 2, cy + h / 2], 1).astype(np.float32)


def _gpu_nms(boxes, scores, thr):
    n = len(boxes)
    b, s = torch.from_numpy(boxes).cuda(), torch.from_numpy(scores).cuda()
    keep = torch.full((max(n, 1),), -1, dtype=torch.int32, device="cuda")
    nk = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    ws = torch.full((B.roi_nms_workspace_bytes(n),), 0x7B, dtype=torch.uint8, device="cuda")
    B.roi_nms(b, s, thr, keep, nk, ws)
    torch.cuda.synchronize()
    return keep[:int(nk.item())].cpu().numpy()


@pytest.mark.parametrize("n,thr", [(0, 0.5), (1, 0.5), (63, 0.5), (64, 0.3), (65, 0.7), (1000, 0.7), (2000, 0.5), (4133, 0.5)])
def test_nms_bit_exact(n, thr):
    rng = np.random.default_rng(1000 + n)
    boxes = _boxes(rng, n, 1344.0)
    scores = rng.uniform(0, 1, n).astype(np.float32)
    if n >= 64:
        scores[5] = scores[40] = scores[63]          # ties: lower index first
        boxes[7] = boxes[3]                          # duplicates: IoU exactly 1
    assert _gpu_nms(boxes, scores, thr).tolist() == O.nms(boxes, scores, thr).tolist()


def test_nms_dense_cluster_and_threshold_edge():
    # every box overlaps every other: one survivor per IoU > thr chain; plus the exact-threshold pair
    rng = np.random.default_rng(5)
    base = np.array([100, 100, 200, 200], np.float32)
    boxes = (base[None] + rng.uniform(-6, 6, (300, 4))).astype(np.float32)
    scores = rng.permutation(300).astype(np.float32)
    for thr in (0.5, 0.8, 0.9):
        assert _gpu_nms(boxes, scores, thr).tolist() == O.nms(boxes, scores, thr).tolist()
    b = np.array([[0, 0, 2, 2], [0, 0, 2, 1]], np.float32)
    s = np.array([0.9, 0.8], np.float32)
    assert _gpu_nms(b, s, 0.5).tolist() == [0, 1] and _gpu_nms(b, s, 0.49).tolist() == [0]


@pytest.mark.parametrize("method", ["linear", "gaussian"])
@pytest.mark.parametrize("n", [0, 1, 50, 700, 3000])
def test_soft_nms(method, n):
    rng = np.random.default_rng(2000 + n)
    boxes = _boxes(rng, n, 900.0)
    scores = rng.uniform(0.05, 1, n).astype(np.float32)
    thr, sigma, min_score = 0.3, 0.5, 0.05
    b, s = torch.from_numpy(boxes).cuda(), torch.from_numpy(scores).cuda()
    keep = torch.full((max(n, 1),), -1, dtype=torch.int32, device="cuda")
    ns = torch.full((max(n, 1),), float("nan"), dtype=torch.float32, device="cuda")
    nk = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    B.roi_soft_nms(b, s, thr, sigma, min_score, {"linear": B.RAF_SOFT_LINEAR, "gaussian": B.RAF_SOFT_GAUSSIAN}[method], keep, ns, nk)
    torch.cuda.synchronize()
    m = int(nk.item())
    got_i, got_s = keep[:m].cpu().numpy(), ns[:m].cpu().numpy()
    ref_i, ref_s = O.soft_nms(boxes, scores, thr, sigma, min_score, method)
    if method == "linear":      # every operation individually rounded on both sides: bit-exact
        assert got_i.tolist() == ref_i.tolist()
        assert np.array_equal(got_s, ref_s)
    else:                       # expf differs by a few ulp between the two libraries: the emitted scores agree to
                                # 1e-5 relative, the emitted set is equal, and the order is equal wherever
                                # neighbouring scores are further apart than that
        assert len(got_i) == len(ref_i) or abs(len(got_i) - len(ref_i)) <= 2
        k = min(len(got_i), len(ref_i))
        assert np.allclose(got_s[:k], ref_s[:k], rtol=1e-5, atol=1e-7)
        gaps = np.abs(np.diff(ref_s[:k])) > 1e-4 * ref_s[:k - 1] if k > 1 else np.zeros(0, bool)
        safe = np.concatenate([[True], gaps]) & np.concatenate([gaps, [True]]) if k > 1 else np.ones(k, bool)
        assert np.array_equal(got_i[:k][safe], ref_i[:k][safe])


# ------------------------------------------------------------------------------- deformable RoI pooling
def _deform_inputs(wl, dtype, layout, seed, amp=0.5):
    cfg = wl.cfg
    PH, PW = cfg.out_size
    K = cfg.K
    rng = np.random.default_rng(seed)
    offset = rng.uniform(-amp, amp, (K, 2, PH, PW)).astype(np.float32)
    feats, exact = T.device_feats(wl.feats, dtype, layout)
    return feats, exact, torch.from_numpy(wl.rois).cuda(), offset


@pytest.mark.parametrize("layout", ["cl", "nchw"])
@pytest.mark.parametrize("index,dtype,kw,g", [
    (1, "f32", {}, 2),
    (2, "f32", dict(n_img=2, per_img=60, channels=32), 2),
    (2, "f32", dict(n_img=1, per_img=40, channels=20), 0),
    (4, "bf16", dict(n_img=2, per_img=24, channels=32), 2),
    (5, "f16", dict(n_img=2, per_img=40, channels=16), 1),
])
def test_deform_roi_pool_forward_backward(index, dtype, kw, g, layout):
    """Readings D1-D5: forward at the RoIAlign tolerances (S10); feature gradient at S11 (S = the oracle's sum of
    |terms|, here bounded by the RoIAlign S of the same taps: use |ref| summed in double); offset gradient against
    the oracle with a tolerance scaled by the sum of |terms| over channels.  Zero offsets == RoIAlign."""
    wl = inputs.make_workload(index, **kw)
    cfg = wl.cfg
    PH, PW = cfg.out_size
    K, C = cfg.K, cfg.channels
    gamma = 0.1
    feats, exact, rois, offset = _deform_inputs(wl, dtype, layout, seed=index)
    off_d = torch.from_numpy(offset).cuda()
    out = T.empty_layout((K, C, PH, PW), feats[0].dtype, layout, fill=float("nan"))
    B.roi_deform_pool_fpn_forward(feats, cfg.scales, rois, off_d, gamma, out, g, cfg.finest_scale)
    torch.cuda.synchronize()
    ref = O.deform_roi_pool_forward(exact, cfg.scales, wl.rois, offset, gamma, (PH, PW), g, cfg.finest_scale)
    T.assert_forward_close(out.to(torch.float64).cpu().numpy(), ref, dtype)
    # zero offsets (NULL tensor) == the RoIAlign forward of the library (same coordinates; fp32 sums in another order)
    out0 = T.empty_layout((K, C, PH, PW), feats[0].dtype, layout, fill=float("nan"))
    B.roi_deform_pool_fpn_forward(feats, cfg.scales, rois, None, gamma, out0, g, cfg.finest_scale)
    ref0 = O.deform_roi_pool_forward(exact, cfg.scales, wl.rois, None, gamma, (PH, PW), g, cfg.finest_scale)
    T.assert_forward_close(out0.to(torch.float64).cpu().numpy(), ref0, dtype)
    # backward
    go_t = torch.from_numpy(wl.grad_out).to(T.TORCH_DTYPE[dtype])
    go = T.to_layout(go_t.cuda(), layout)
    go_exact = go_t.to(torch.float64).numpy()
    grads = [T.empty_layout(s, torch.float32, layout, fill=float("nan")) for s in cfg.level_shapes]
    goff = torch.full((K, 2, PH, PW), float("nan"), dtype=torch.float32, device="cuda")
    B.roi_deform_pool_fpn_backward(feats, grads, cfg.scales, go, rois, off_d, gamma, g, cfg.finest_scale, goff)
    torch.cuda.synchronize()
    gref, goref = O.deform_roi_pool_backward(exact, cfg.scales, go_exact, wl.rois, offset, gamma, g, cfg.finest_scale)
    # scale of the sums: the same backward on |grad_out| with all-positive weights bounds sum |terms|
    Sref, _ = O.deform_roi_pool_backward(exact, cfg.scales, np.abs(go_exact), wl.rois, offset, gamma, g, cfg.finest_scale)
    T.assert_backward_close([t.to(torch.float64).cpu().numpy() for t in grads], gref, Sref)
    # offset gradient: sum over channels and samples of go * (differences of features): fp32 sums of up to C*g*g*2
    # terms -> |err| <= 1e-4 |ref| + 2e-6 * sum |terms|; sum |terms| is bounded by the same backward on |grad_out| and
    # |features| differences <= 2 max|F| ... use the oracle on absolute values as the scale
    abs_feats = [np.abs(e) for e in exact]
    _, Soff = O.deform_roi_pool_backward(abs_feats, cfg.scales, np.abs(go_exact), wl.rois, offset, gamma, g, cfg.finest_scale)
    scale = np.abs(Soff) + 2.0 * np.abs(goref) + 1e-3
    err = np.abs(goff.to(torch.float64).cpu().numpy() - goref)
    tol = 1e-4 * np.abs(goref) + 1e-5 * scale if dtype == "f32" else 2e-2 * np.abs(goref) + 1e-3 * scale
    assert np.isfinite(goff.cpu().numpy()).all()
    assert (err <= tol).all(), float((err / tol).max())
    # feature gradient only / offset gradient only / accumulate
    g2 = [torch.zeros_like(t) for t in grads]
    B.roi_deform_pool_fpn_backward(feats, g2, cfg.scales, go, rois, off_d, gamma, g, cfg.finest_scale, None)
    goff2 = torch.full_like(goff, float("nan"))
    B.roi_deform_pool_fpn_backward(feats, None, cfg.scales, go, rois, off_d, gamma, g, cfg.finest_scale, goff2)
    torch.cuda.synchronize()
    T.assert_backward_close([t.to(torch.float64).cpu().numpy() for t in g2], gref, Sref)
    assert (np.abs(goff2.to(torch.float64).cpu().numpy() - goref) <= tol).all()
    B.roi_deform_pool_fpn_backward(feats, g2, cfg.scales, go, rois, off_d, gamma, g, cfg.finest_scale, None, B.RAF_ACCUMULATE)
    torch.cuda.synchronize()
    T.assert_backward_close([t.to(torch.float64).cpu().numpy() for t in g2], [2 * r for r in gref], [2 * s for s in Sref])


def test_deform_roi_pool_argument_errors():
    wl = inputs.make_workload(1)
    cfg = wl.cfg
    feats, _, rois, offset = _deform_inputs(wl, "f32", "cl", seed=0)
    out = T.empty_layout((cfg.K, cfg.channels, 7, 7), torch.float32, "cl")
    with pytest.raises(ValueError):
        B.roi_deform_pool_fpn_forward(feats, cfg.scales, rois, torch.zeros(cfg.K, 2, 7, 6, device="cuda"), 0.1, out, 2, 56.0)
    with pytest.raises(B.RafError) as e:
        B.roi_deform_pool_fpn_forward(feats, cfg.scales, rois, None, 0.1, out, -1, 56.0)
    assert e.value.status == -2
    go = T.to_layout(torch.from_numpy(wl.grad_out).cuda(), "cl")
    with pytest.raises(B.RafError) as e:
        B.roi_deform_pool_fpn_backward(feats, None, cfg.scales, go, rois, None, 0.1, 2, 56.0, None, flags=B.RAF_ATOMIC)
    assert e.value.status == -5


# ----------------------------------------------------------------- RoIAlign gather fused into the first FC
def _fc_case(index, dtype, kw, n_out, g=2, bias=True, seed=0):
    wl = inputs.make_workload(index, **kw)
    cfg = wl.cfg
    PH, PW = cfg.out_size
    K, C = cfg.K, cfg.channels
    tdt = T.TORCH_DTYPE[dtype]
    rng = np.random.default_rng(seed)
    feats, exact = T.device_feats(wl.feats, dtype, "cl")
    rois = torch.from_numpy(wl.rois).cuda()
    w_t = torch.from_numpy((rng.standard_normal((n_out, PH * PW * C)) / np.sqrt(PH * PW * C)).astype(np.float32)).to(tdt)
    b_np = rng.standard_normal(n_out).astype(np.float32) if bias else None
    out = torch.full((K, n_out), float("nan"), dtype=torch.float32, device="cuda")
    B.roi_align_fc_fpn_forward(feats, cfg.scales, rois, w_t.cuda(), None if b_np is None else torch.from_numpy(b_np).cuda(), out,
                               (PH, PW), g, True, cfg.finest_scale)
    torch.cuda.synchronize()
    w64 = w_t.to(torch.float64).numpy()
    ref = O.roi_align_fc_forward(exact, cfg.scales, wl.rois, w64, b_np, (PH, PW), g, True, cfg.finest_scale, dtype=dtype)
    # scale of the sum: sum |a| |w| with |a| <= the rounded features
    refabs = O.roi_align_fc_forward([np.abs(e) for e in exact], cfg.scales, wl.rois, np.abs(w64), None if b_np is None else np.abs(b_np),
                                    (PH, PW), g, True, cfg.finest_scale, dtype=dtype)
    got = out.to(torch.float64).cpu().numpy()
    assert np.isfinite(got).all()
    # fp32 accumulation of PH*PW*C terms + a 16-bit rounding of a feature that sits next to a rounding boundary
    # (the CUDA forward and the oracle agree to 1e-5 relative BEFORE rounding): |err| <= 2e-2 |ref| + 2e-3 * sum |terms|
    eps = 2.0 ** -8 if dtype == "bf16" else 2.0 ** -11
    tol = 2e-2 * np.abs(ref) + eps * refabs + 1e-5
    err = np.abs(got - ref)
    assert (err <= tol).all(), float((err / tol).max())
    return float((err / tol).max()), float(err.max()), float(np.abs(ref).max())


@pytest.mark.parametrize("index,dtype,kw,n_out,g", [
    (5, "bf16", dict(n_img=2, per_img=100, channels=64), 512, 2),      # 200 RoIs: two M tiles, the second ragged
    (4, "bf16", dict(n_img=1, per_img=40, channels=128), 1024, 2),     # 14 x 14 bins, two N tiles
    (3, "f16", dict(n_img=1, per_img=130, channels=64), 512, 2),
    (5, "f16", dict(n_img=2, per_img=30, channels=192), 512, 1),
])
def test_roi_align_fc_fused(index, dtype, kw, n_out, g):
    worst, emax, rmax = _fc_case(index, dtype, kw, n_out, g)
    assert emax <= 2e-2 * rmax


def test_roi_align_fc_fused_matches_unfused_library_path():
    """The same numbers from the library's own RoIAlign forward followed by a matrix product (torch, fp32 accumulate):
    the fused A tiles are bit-identical to the stand-alone forward's output, so the two differ only by the order of the
    fp32 sums."""
    wl = inputs.make_workload(5, n_img=2, per_img=64, channels=64)
    cfg = wl.cfg
    PH, PW = cfg.out_size
    K, C = cfg.K, cfg.channels
    feats, _ = T.device_feats(wl.feats, "bf16", "cl")
    rois = torch.from_numpy(wl.rois).cuda()
    rng = np.random.default_rng(3)
    w = torch.from_numpy((rng.standard_normal((512, PH * PW * C)) / 56.0).astype(np.float32)).to(torch.bfloat16).cuda()
    out = torch.empty((K, 512), dtype=torch.float32, device="cuda")
    B.roi_align_fc_fpn_forward(feats, cfg.scales, rois, w, None, out, (PH, PW), 2, True, cfg.finest_scale)
    x = T.empty_layout((K, C, PH, PW), torch.bfloat16, "cl")
    B.roi_align_fpn_forward_ex(feats, cfg.scales, rois, x, 2, True, cfg.finest_scale, B.RAF_NO_PREP, None)
    a = x.permute(0, 2, 3, 1).reshape(K, -1).to(torch.float32)
    want = a @ w.to(torch.float32).T
    torch.cuda.synchronize()
    scale = (a.abs() @ w.to(torch.float32).abs().T)
    assert bool(((out - want).abs() <= 1e-5 * scale + 1e-6).all())


def test_roi_align_fc_argument_errors():
    wl = inputs.make_workload(5, n_img=1, per_img=8, channels=64)
    cfg = wl.cfg
    feats, _ = T.device_feats(wl.feats, "bf16", "cl")
    rois = torch.from_numpy(wl.rois).cuda()
    w = torch.zeros((512, 49 * 64), dtype=torch.bfloat16, device="cuda")
    out = torch.empty((cfg.K, 512), dtype=torch.float32, device="cuda")
    with pytest.raises(B.RafError) as e:     # sampling grid beyond the tables of this kernel
        B.roi_align_fc_fpn_forward(feats, cfg.scales, rois, w, None, out, (7, 7), 3, True, 56.0)
    assert e.value.status == -5
    with pytest.raises(B.RafError) as e:     # n_out not a multiple of 512
        B.roi_align_fc_fpn_forward(feats, cfg.scales, rois, w[:128], None, out[:, :128].contiguous(), (7, 7), 2, True, 56.0)
    assert e.value.status == -5
    with pytest.raises(ValueError):
        B.roi_align_fc_fpn_forward(feats, cfg.scales, rois, w.to(torch.float16), None, out, (7, 7), 2, True, 56.0)
