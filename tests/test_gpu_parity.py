"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Level assignment / bucketing bit-exact; forward and backward within the
tolerances of readings S10 / S11 (BASELINE.json north_star)."""
import numpy as np
import pytest
import torch

from oracle import raf_ref as R
from paper_1906_07155_b200 import binding as B
from paper_1906_07155_b200 import inputs
import raf_testlib as T

pytestmark = pytest.mark.gpu


# ------------------------------------------------------------------------------------------------
# K1: levels / histogram / stable bucketing -- bit exact
# ------------------------------------------------------------------------------------------------
def _gpu_levels(rois_np, L, fs):
    K = rois_np.shape[0]
    rois = torch.from_numpy(np.ascontiguousarray(rois_np, np.float32)).cuda()
    levels = torch.full((max(K, 1),), -7, dtype=torch.int32, device="cuda")
    counts = torch.full((L,), -7, dtype=torch.int32, device="cuda")
    perm = torch.full((max(K, 1),), -7, dtype=torch.int32, device="cuda")
    B.roi_fpn_assign_levels(rois, L, fs, levels, counts, perm)
    torch.cuda.synchronize()
    return levels[:K].cpu().numpy(), counts.cpu().numpy(), perm[:K].cpu().numpy()


@pytest.mark.parametrize("index", [2, 3, 4, 5])
def test_levels_bit_exact_configs(index):
    wl = inputs.make_workload(index, with_feats=False, with_grad=False)
    got = _gpu_levels(wl.rois, 4, 56.0)
    ref = R.assign_levels(wl.rois, 4, 56.0)
    for g, r in zip(got, ref):
        assert np.array_equal(g, r)
    assert got[1].tolist() == list(wl.cfg.level_hist)


@pytest.mark.parametrize("L,fs", [(4, 56.0), (1, 56.0), (2, 56.0), (8, 7.0), (5, 33.3)])
def test_levels_bit_exact_adversarial(L, fs):
    rois = inputs.adversarial_level_rois(fs, min(L, 6))
    rng = np.random.default_rng(1)
    rois = rois[rng.permutation(len(rois))]          # shuffled: stability must not rely on order
    got = _gpu_levels(rois, L, fs)
    ref = R.assign_levels(rois, L, fs)
    for g, r in zip(got, ref):
        assert np.array_equal(g, r)


@pytest.mark.parametrize("K", [0, 1, 31, 1024, 1025, 5000])
def test_levels_sizes_and_ragged_tail(K):
    rng = np.random.default_rng(K)
    side = np.exp(rng.uniform(np.log(8), np.log(1500), K))
    rois = np.stack([np.zeros(K), np.zeros(K), np.zeros(K), side, side * rng.uniform(0.5, 2, K)], 1).astype(np.float32)
    got = _gpu_levels(rois, 4, 56.0)
    ref = R.assign_levels(rois, 4, 56.0)
    for g, r in zip(got, ref):
        assert np.array_equal(g, r)


# ------------------------------------------------------------------------------------------------
# K2 forward
# ------------------------------------------------------------------------------------------------
def _fwd_case(wl, dtype, layout, P=None, g=None, aligned=None):
    cfg = wl.cfg
    P = P or cfg.out_size
    g = cfg.sampling_ratio if g is None else g
    aligned = cfg.aligned if aligned is None else aligned
    dev, exact = T.device_feats(wl.feats, dtype, layout)
    got = T.gpu_forward(dev, cfg.scales, wl.rois, P, g, aligned, cfg.finest_scale, layout)
    ref = R.forward(exact, cfg.scales, wl.rois, P, g, aligned, cfg.finest_scale, coord_f32=True)
    return T.assert_forward_close(got, ref, dtype)


@pytest.mark.parametrize("layout", ["cl", "nchw"])
def test_forward_config1(layout):
    _fwd_case(inputs.make_workload(1), "f32", layout)


@pytest.mark.parametrize("layout", ["cl", "nchw"])
@pytest.mark.parametrize("index,dtype,kw", [
    (2, "f32", dict(n_img=2, per_img=96)),
    (3, "f16", dict(n_img=1, per_img=150)),
    (4, "bf16", dict(n_img=2, per_img=40)),
    (5, "bf16", dict(n_img=3, per_img=64)),     # boxes partly outside the image
    (5, "f32", dict(n_img=2, per_img=50, channels=36)),   # C not a multiple of 32 lanes
])
def test_forward_reduced_configs(index, dtype, kw, layout):
    _fwd_case(inputs.make_workload(index, **kw), dtype, layout)


@pytest.mark.parametrize("layout", ["cl", "nchw"])
@pytest.mark.parametrize("P,g,aligned", [((7, 7), 1, True), ((7, 7), 3, True), ((7, 7), 0, True),
                                         ((7, 7), 2, False), ((7, 7), 0, False), ((5, 9), 2, True),
                                         ((1, 1), 4, True), ((14, 14), 2, False), ((32, 32), 2, True),
                                         ((3, 2), 16, True)])
def test_forward_variants(P, g, aligned, layout):
    wl = inputs.make_workload(5, n_img=2, per_img=24, channels=8)
    _fwd_case(wl, "f32", layout, P=P, g=g, aligned=aligned)


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_adaptive_large_grids_forward_and_backward(dtype):
    """sampling_ratio = 0 with bins of up to ~30 pixels (grids far beyond the 8 x 8 the forward tabulates: its
    sample-by-sample path) next to small boxes (grid 1) and boxes with no extent (grid 0, reading S7), on one
    60 x 70 map: forward, and the deterministic strip backward with its per-RoI grids."""
    rng = np.random.default_rng(21)
    K, C, H, W = 40, 24, 60, 70
    side = np.exp(rng.uniform(np.log(0.5), np.log(220.0), (K, 2)))
    cx, cy = rng.uniform(-5, W + 5, K), rng.uniform(-5, H + 5, K)
    rois = np.stack([np.zeros(K), cx - side[:, 0] / 2, cy - side[:, 1] / 2, cx + side[:, 0] / 2,
                     cy + side[:, 1] / 2], 1).astype(np.float32)
    rois[3, 3] = rois[3, 1]            # zero width: gw = 0 -> no samples
    rois[5, 2], rois[5, 4] = rois[5, 4], rois[5, 2]   # reversed rows
    feats = [rng.standard_normal((1, C, H, W)).astype(np.float32)]
    dev, exact = T.device_feats(feats, dtype, "cl")
    got = T.gpu_forward(dev, [1.0], rois, (7, 7), 0, True, 56.0, "cl")
    ref = R.forward(exact, [1.0], rois, (7, 7), 0, True, 56.0, coord_f32=True)
    T.assert_forward_close(got, ref, dtype)
    gout = rng.standard_normal((K, C, 7, 7)).astype(np.float32)
    for flags in (0, B.RAF_DETERMINISTIC, B.RAF_ATOMIC):
        gg, go_exact = T.gpu_backward([(1, C, H, W)], [1.0], gout, rois, 0, True, 56.0, "cl", dtype, flags)
        gref, S = R.backward([(1, C, H, W)], [1.0], go_exact, rois, (7, 7), 0, True, 56.0)
        T.assert_backward_close(gg, gref, S)


def test_forward_degenerate_and_invalid_rois():
    wl = inputs.make_workload(2, n_img=2, per_img=8, channels=16)
    rois = np.array([[0, 100, 100, 100, 100], [1, 300, 200, 100, 50], [0, -500, -500, -400, -400],
                     [1, 0, 0, 1344, 800], [2, 10, 10, 90, 90], [-1, 10, 10, 90, 90],
                     [0.5, 10, 10, 90, 90], [0, 1343.9, 799.9, 1344, 800], [1, 5000, 5000, 6000, 6000]], np.float32)
    wl.rois = rois
    for layout in ("cl", "nchw"):
        dev, exact = T.device_feats(wl.feats, "f32", layout)
        got = T.gpu_forward(dev, wl.cfg.scales, rois, (7, 7), 2, True, 56.0, layout)
        ref = R.forward(exact, wl.cfg.scales, rois, (7, 7), 2, True, 56.0, coord_f32=True)
        T.assert_forward_close(got, ref, "f32")
        assert np.all(got[4:7] == 0)     # invalid batch index -> zero rows (reading S17)


def test_forward_metamorphic_layouts_and_permutation():
    wl = inputs.make_workload(2, n_img=2, per_img=64, channels=64)
    cfg = wl.cfg
    outs = {}
    for layout in ("cl", "nchw"):
        dev, _ = T.device_feats(wl.feats, "f32", layout)
        outs[layout] = T.gpu_forward(dev, cfg.scales, wl.rois, (7, 7), 2, True, 56.0, layout)
    # same coordinates and weights in both kernels; only the accumulation order may differ
    assert np.abs(outs["cl"] - outs["nchw"]).max() < 2e-6
    p = np.random.default_rng(0).permutation(cfg.K)
    dev, _ = T.device_feats(wl.feats, "f32", "cl")
    shuffled = T.gpu_forward(dev, cfg.scales, wl.rois[p], (7, 7), 2, True, 56.0, "cl")
    assert np.array_equal(shuffled, outs["cl"][p])
    # channel slicing: a strided channel slice of the channels-last buffer (generic path) agrees
    dev_slice = [d[:, 8:24] for d in dev]
    sl = T.gpu_forward(dev_slice, cfg.scales, wl.rois, (7, 7), 2, True, 56.0, "cl")
    assert np.abs(sl - outs["cl"][:, 8:24]).max() < 2e-6


@pytest.mark.parametrize("index", [2, 3, 4, 5])
def test_forward_full_size_sampled(index):
    """BASELINE.json full sizes in the layout bench.py times; the oracle recomputes a sample of RoIs
    (rows are independent, so row k of the full run must equal the oracle on rois[k])."""
    wl = inputs.make_workload(index, with_grad=False)
    cfg = wl.cfg
    dev, _ = T.device_feats(wl.feats, cfg.dtype, "cl")
    got = T.gpu_forward(dev, cfg.scales, wl.rois, cfg.out_size, 2, True, 56.0, "cl")
    assert np.isfinite(got).all()
    rng = np.random.default_rng(index)
    pick = np.sort(rng.choice(cfg.K, 48, replace=False))
    exact = [d.permute(0, 1, 2, 3).to(torch.float64).cpu().numpy() for d in dev]
    ref = R.forward(exact, cfg.scales, wl.rois[pick], cfg.out_size, 2, True, 56.0, coord_f32=True)
    T.assert_forward_close(got[pick], ref, cfg.dtype)


# ------------------------------------------------------------------------------------------------
# K3 backward
# ------------------------------------------------------------------------------------------------
def _bwd_case(wl, gout_dtype, layout, P=None, g=None, aligned=None, flags=0, init=None):
    cfg = wl.cfg
    P = P or cfg.out_size
    g = cfg.sampling_ratio if g is None else g
    aligned = cfg.aligned if aligned is None else aligned
    gout = wl.grad_out
    if gout.shape[2:] != tuple(P):
        gout = np.random.default_rng(5).standard_normal((cfg.K, cfg.channels, *P)).astype(np.float32)
    got, go_exact = T.gpu_backward(cfg.level_shapes, cfg.scales, gout, wl.rois, g, aligned, cfg.finest_scale,
                                   layout, gout_dtype, flags, init)
    ref, S = R.backward(cfg.level_shapes, cfg.scales, go_exact, wl.rois, P, g, aligned, cfg.finest_scale,
                        coord_f32=True, accumulate_into=init)
    if init is not None:   # starting values count towards the error scale
        S = [s + np.abs(i) for s, i in zip(S, init)]
    return T.assert_backward_close(got, ref, S)


VARIANTS = [("cl", 0), ("cl", B.RAF_ATOMIC), ("cl", B.RAF_DETERMINISTIC), ("cl", B.RAF_PULL_STRIP),
            ("cl", B.RAF_PULL_TILE), ("nchw", 0)]


@pytest.mark.parametrize("layout,flags", VARIANTS)
def test_backward_config1(layout, flags):
    _bwd_case(inputs.make_workload(1), "f32", layout, flags=flags)


@pytest.mark.parametrize("layout,flags", VARIANTS)
@pytest.mark.parametrize("index,dtype,kw", [
    (2, "f32", dict(n_img=2, per_img=96, channels=64)),
    (2, "f32", dict(n_img=1, per_img=300, channels=256)),   # one big (level, image) bucket, full 256-channel chunk
    (4, "bf16", dict(n_img=2, per_img=40, channels=32)),
    (5, "bf16", dict(n_img=3, per_img=64, channels=32)),
    (5, "f16", dict(n_img=2, per_img=50, channels=36)),
    (5, "f32", dict(n_img=2, per_img=30, channels=1040)),   # more channel groups than threads per row
])
def test_backward_reduced_configs(index, dtype, kw, layout, flags):
    _bwd_case(inputs.make_workload(index, **kw), dtype, layout, flags=flags)


@pytest.mark.parametrize("layout,flags", [("cl", 0), ("cl", B.RAF_ATOMIC), ("cl", B.RAF_PULL_STRIP),
                                          ("cl", B.RAF_DETERMINISTIC), ("nchw", 0)])
@pytest.mark.parametrize("P,g,aligned", [((7, 7), 1, True), ((7, 7), 0, True), ((7, 7), 2, False),
                                         ((5, 9), 3, True), ((14, 14), 2, True), ((7, 7), 0, False),
                                         ((32, 32), 2, True), ((1, 1), 4, True), ((3, 2), 16, False)])
def test_backward_variants(P, g, aligned, layout, flags):
    wl = inputs.make_workload(5, n_img=2, per_img=24, channels=8)
    _bwd_case(wl, "f32", layout, P=P, g=g, aligned=aligned, flags=flags)


def _single_level_case(K, C, H, W, side_lo, side_hi, seed, flags, P=(7, 7), g=2, dtype="f32"):
    """Many RoIs on ONE small map: exercises the pull kernel's multi-pass tiles (more than 16
    candidates per tile), scan chunks (more than 512 RoIs per bucket) and, with tiny boxes, the
    slow path (more than two tap entries per pixel row / column)."""
    rng = np.random.default_rng(seed)
    side = rng.uniform(side_lo, side_hi, (K, 2))
    cx, cy = rng.uniform(-1, W + 1, K), rng.uniform(-1, H + 1, K)
    rois = np.stack([np.zeros(K), cx - side[:, 0] / 2, cy - side[:, 1] / 2, cx + side[:, 0] / 2,
                     cy + side[:, 1] / 2], 1).astype(np.float32)
    gout = rng.standard_normal((K, C, *P)).astype(np.float32)
    shapes, scales = [(1, C, H, W)], [1.0]
    got, go_exact = T.gpu_backward(shapes, scales, gout, rois, g, True, 56.0, "cl", dtype, flags)
    ref, S = R.backward(shapes, scales, go_exact, rois, P, g, True, 56.0)
    return T.assert_backward_close(got, ref, S)


@pytest.mark.parametrize("flags", [0, B.RAF_DETERMINISTIC, B.RAF_ATOMIC, B.RAF_PULL_STRIP, B.RAF_PULL_TILE])
def test_backward_dense_tiles_and_big_buckets(flags):
    _single_level_case(K=700, C=16, H=24, W=40, side_lo=4, side_hi=20, seed=11, flags=flags)


@pytest.mark.parametrize("flags", [0, B.RAF_ATOMIC, B.RAF_PULL_STRIP])
@pytest.mark.parametrize("C,dtype", [(8, "f32"), (320, "f32"), (264, "bf16")])
def test_backward_tiny_boxes_many_entries_per_pixel(flags, C, dtype):
    # boxes of 0.3 .. 3 px: bins narrower than half a pixel -> up to 7 entries per row / column
    _single_level_case(K=90, C=C, H=17, W=19, side_lo=0.3, side_hi=3.0, seed=12, flags=flags, dtype=dtype)


@pytest.mark.parametrize("P,g", [((14, 14), 2), ((9, 20), 3)])
@pytest.mark.parametrize("flags", [B.RAF_PULL_TILE, B.RAF_PULL_STRIP])
def test_backward_many_taps_dense(P, g, flags):
    # more than 32 taps per axis (two / four ballot chunks of the tile kernel) on a dense map
    _single_level_case(K=120, C=12, H=20, W=20, side_lo=2, side_hi=18, seed=13, flags=flags, P=P, g=g)


@pytest.mark.parametrize("flags", [0, B.RAF_DETERMINISTIC, B.RAF_PULL_STRIP])
def test_backward_largest_output_and_grid(flags):
    # 32 x 32 bins with a 4 x 4 sampling grid (256 sample taps per axis): the largest output the ABI takes;
    # the strip backward's dense per-bin weights have no tap-count limit, so this is deterministic too
    _single_level_case(K=20, C=8, H=20, W=20, side_lo=2, side_hi=18, seed=14, flags=flags, P=(32, 32), g=4)


@pytest.mark.parametrize("variant", [B.RAF_PULL_TILE, B.RAF_PULL_STRIP])
@pytest.mark.parametrize("layout_fwd", ["cl", "nchw"])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_backward_reuses_prep_written_by_forward(layout_fwd, dtype, variant):
    """RAF_REUSE_PREP: the forward call leaves the RoI buckets / tap tables in the workspace (in the
    leading blocks of its own launch for channels-last, by a separate launch otherwise); the backward
    skips its prep launch.  Result must equal the oracle and the stand-alone backward bit for bit."""
    wl = inputs.make_workload(5, n_img=3, per_img=120, channels=64)
    cfg = wl.cfg
    PH, PW = cfg.out_size
    K, C, L = cfg.K, cfg.channels, len(cfg.level_shapes)
    feats, _ = T.device_feats(wl.feats, dtype, layout_fwd)
    rois = torch.from_numpy(wl.rois).cuda()
    go_t = torch.from_numpy(wl.grad_out).to(T.TORCH_DTYPE[dtype])
    go = T.to_layout(go_t.cuda(), "cl")
    ws = T.workspace(K, L, PH, PW, 2)
    ws.fill_(0xAB)
    out = T.empty_layout((K, C, PH, PW), feats[0].dtype, layout_fwd)
    B.roi_align_fpn_forward(feats, cfg.scales, rois, out, 2, True, cfg.finest_scale, ws)
    g1 = [T.empty_layout(s, torch.float32, "cl", fill=float("nan")) for s in cfg.level_shapes]
    B.roi_align_fpn_backward(g1, cfg.scales, go, rois, 2, True, cfg.finest_scale, B.RAF_REUSE_PREP | variant, ws)
    torch.cuda.synchronize()
    ws2 = T.workspace(K, L, PH, PW, 2)
    g2 = [T.empty_layout(s, torch.float32, "cl", fill=float("nan")) for s in cfg.level_shapes]
    B.roi_align_fpn_backward(g2, cfg.scales, go, rois, 2, True, cfg.finest_scale, variant, ws2)
    torch.cuda.synchronize()
    for a_, b_ in zip(g1, g2):
        assert torch.equal(a_, b_)
    ref, S = R.backward(cfg.level_shapes, cfg.scales, go_t.to(torch.float64).numpy(), wl.rois, (PH, PW), 2, True,
                        cfg.finest_scale)
    T.assert_backward_close([t.to(torch.float64).cpu().numpy() for t in g1], ref, S)


def test_backward_degenerate_and_invalid_rois():
    wl = inputs.make_workload(2, n_img=2, per_img=8, channels=16)
    wl.rois = np.array([[0, 100, 100, 100, 100], [1, 300, 200, 100, 50], [0, -500, -500, -400, -400],
                        [1, 0, 0, 1344, 800], [2, 10, 10, 90, 90], [-1, 10, 10, 90, 90],
                        [0.5, 10, 10, 90, 90], [0, 1343.9, 799.9, 1344, 800], [1, 5000, 5000, 6000, 6000],
                        [0, -3, -3, 2, 2], [1, 1340, 790, 1350, 810]], np.float32)
    wl.grad_out = wl.grad_out[:len(wl.rois)]
    for layout, flags in VARIANTS:
        cfg = wl.cfg
        got, go_exact = T.gpu_backward(cfg.level_shapes, cfg.scales, wl.grad_out, wl.rois, 2, True, 56.0, layout,
                                       "f32", flags)
        ref, S = R.backward(cfg.level_shapes, cfg.scales, go_exact, wl.rois, (7, 7), 2, True, 56.0)
        T.assert_backward_close(got, ref, S)


@pytest.mark.parametrize("variant", [0, B.RAF_PULL_STRIP, B.RAF_PULL_TILE])
def test_deterministic_backward_is_bit_reproducible(variant):
    wl = inputs.make_workload(5, n_img=3, per_img=200, channels=64)
    cfg = wl.cfg
    runs = [T.gpu_backward(cfg.level_shapes, cfg.scales, wl.grad_out, wl.rois, 2, True, 56.0, "cl", "bf16",
                           B.RAF_DETERMINISTIC | variant)[0] for _ in range(3)]
    for other in runs[1:]:
        for a, b in zip(runs[0], other):
            assert np.array_equal(a, b)
    # requesting determinism for an ineligible layout is refused, not silently downgraded
    with pytest.raises(B.RafError) as e:
        T.gpu_backward(cfg.level_shapes, cfg.scales, wl.grad_out, wl.rois, 2, True, 56.0, "nchw", "f32",
                       B.RAF_DETERMINISTIC)
    assert e.value.status == -5


@pytest.mark.parametrize("layout,flags", VARIANTS)
def test_backward_accumulate_mode(layout, flags):
    wl = inputs.make_workload(2, n_img=2, per_img=32, channels=16)
    rng = np.random.default_rng(3)
    init = [rng.standard_normal(s).astype(np.float32).astype(np.float64) for s in wl.cfg.level_shapes]
    _bwd_case(wl, "f32", layout, flags=flags | B.RAF_ACCUMULATE, init=init)


@pytest.mark.parametrize("flags", [0, B.RAF_ATOMIC, B.RAF_PULL_STRIP])
def test_backward_full_size_config2(flags):
    wl = inputs.make_workload(2, with_feats=False)
    cfg = wl.cfg
    got, go_exact = T.gpu_backward(cfg.level_shapes, cfg.scales, wl.grad_out, wl.rois, 2, True, 56.0, "cl",
                                   "f32", flags)
    # the oracle on two channel slices, one in each 128-channel half of a lane's accumulators
    # (channels are independent)
    shapes = [(s[0], 16, s[2], s[3]) for s in cfg.level_shapes]
    for sl in (slice(40, 56), slice(224, 240)):
        ref, S = R.backward(shapes, cfg.scales, go_exact[:, sl], wl.rois, (7, 7), 2, True, 56.0)
        T.assert_backward_close([g[:, sl] for g in got], ref, S)
    # properties that hold at any size: total mass and untouched pixels
    masks = R.footprint(cfg.level_shapes, cfg.scales, wl.rois, (7, 7), 2, True)
    for g, m in zip(got, masks):
        assert np.all(g[np.broadcast_to(m[:, None] == 0, g.shape)] == 0)


@pytest.mark.parametrize("index", [2, 4, 5])
def test_full_size_step_as_benched(index):
    """BASELINE.json full sizes in exactly the launch configuration bench.py times: channels-last,
    forward first, then the backward with RAF_REUSE_PREP on the same workspace (two launches per
    step).  Forward: sampled rows against the oracle.  Backward: a 16-channel slice against the
    oracle (channels are independent), plus properties that hold at any size (untouched pixels
    exactly zero, every element finite) on all channels."""
    wl = inputs.make_workload(index)
    cfg = wl.cfg
    tdt = T.TORCH_DTYPE[cfg.dtype]
    PH, PW = cfg.out_size
    K, C, L = cfg.K, cfg.channels, len(cfg.level_shapes)
    feats, _ = T.device_feats(wl.feats, cfg.dtype, "cl")
    rois = torch.from_numpy(wl.rois).cuda()
    out = T.empty_layout((K, C, PH, PW), tdt, "cl", fill=float("nan"))
    go_t = torch.from_numpy(wl.grad_out).to(tdt)
    gout = T.to_layout(go_t.cuda(), "cl")
    grads = [T.empty_layout(s_, torch.float32, "cl", fill=float("nan")) for s_ in cfg.level_shapes]
    ws = T.workspace(K, L, PH, PW, 2, B.RAF_REUSE_PREP)
    B.roi_align_fpn_forward(feats, cfg.scales, rois, out, 2, True, cfg.finest_scale, ws)
    B.roi_align_fpn_backward(grads, cfg.scales, gout, rois, 2, True, cfg.finest_scale, B.RAF_REUSE_PREP, ws)
    torch.cuda.synchronize()
    # forward, sampled rows
    pick = np.sort(np.random.default_rng(100 + index).choice(K, 32, replace=False))
    exact = [f.to(torch.float64).cpu().numpy() for f in feats]
    ref = R.forward(exact, cfg.scales, wl.rois[pick], (PH, PW), 2, True, cfg.finest_scale)
    T.assert_forward_close(out[torch.from_numpy(pick).cuda()].to(torch.float64).cpu().numpy(), ref, cfg.dtype)
    del exact
    # backward, two channel slices (one per 128-channel half)
    shapes = [(s_[0], 16, s_[2], s_[3]) for s_ in cfg.level_shapes]
    for sl in (slice(96, 112), slice(224, 240)):
        gref, S = R.backward(shapes, cfg.scales, go_t[:, sl].to(torch.float64).numpy(), wl.rois, (PH, PW), 2, True,
                             cfg.finest_scale)
        T.assert_backward_close([g[:, sl].to(torch.float64).cpu().numpy() for g in grads], gref, S)
    masks = R.footprint(cfg.level_shapes, cfg.scales, wl.rois, (PH, PW), 2, True)
    for g, m in zip(grads, masks):
        assert bool(torch.isfinite(g).all())
        untouched = torch.from_numpy(m == 0).cuda()[:, None].expand_as(g)
        assert bool((g[untouched] == 0).all())


def test_backward_full_size_config5_atomic():
    """Config 5 at full size through the atomic variant (red.global.add.v4.f32), bf16 grad_out."""
    wl = inputs.make_workload(5, with_feats=False)
    cfg = wl.cfg
    got, go_exact = T.gpu_backward(cfg.level_shapes, cfg.scales, wl.grad_out, wl.rois, 2, True, cfg.finest_scale, "cl",
                                   "bf16", B.RAF_ATOMIC)
    shapes = [(s[0], 8, s[2], s[3]) for s in cfg.level_shapes]
    for sl in (slice(16, 24), slice(200, 208)):
        ref, S = R.backward(shapes, cfg.scales, go_exact[:, sl], wl.rois, (7, 7), 2, True, cfg.finest_scale)
        T.assert_backward_close([g[:, sl] for g in got], ref, S)


@pytest.mark.parametrize("variant", [B.RAF_PULL_TILE, B.RAF_PULL_STRIP])
def test_reuse_prep_with_foreign_workspace_is_loud(variant):
    """RAF_REUSE_PREP on a workspace that was NOT written for these arguments (forward on other RoIs, other
    K, other geometry, or never written at all): the pull kernel compares the fingerprint the prep left and
    poisons the whole gradient pyramid with NaN instead of computing from foreign tables."""
    wl = inputs.make_workload(5, n_img=2, per_img=64, channels=32)
    cfg = wl.cfg
    PH, PW = cfg.out_size
    K, C, L = cfg.K, cfg.channels, len(cfg.level_shapes)
    feats, _ = T.device_feats(wl.feats, "f32", "cl")
    rois = torch.from_numpy(wl.rois).cuda()
    other = rois.clone()                       # same values, another buffer: a different RoI tensor
    go = T.to_layout(torch.from_numpy(wl.grad_out).cuda(), "cl")
    out = T.empty_layout((K, C, PH, PW), torch.float32, "cl")

    def bwd(rois_t, ws, flags, g=2, aligned=True):
        grads = [T.empty_layout(s, torch.float32, "cl", fill=1.0) for s in cfg.level_shapes]
        B.roi_align_fpn_backward(grads, cfg.scales, go, rois_t, g, aligned, cfg.finest_scale, flags | variant, ws)
        torch.cuda.synchronize()
        return grads

    ws = T.workspace(K, L, PH, PW, 2)
    B.roi_align_fpn_forward(feats, cfg.scales, rois, out, 2, True, cfg.finest_scale, ws)
    good = bwd(rois, ws, B.RAF_REUSE_PREP)
    assert all(bool(torch.isfinite(g).all()) for g in good)
    for bad in (bwd(other, ws, B.RAF_REUSE_PREP),                       # forward ran on another RoI tensor
                bwd(rois, ws, B.RAF_REUSE_PREP, aligned=False),         # other geometry
                bwd(rois, T.workspace(K, L, PH, PW, 2), B.RAF_REUSE_PREP)):   # never written
        assert all(bool(torch.isnan(g).all()) for g in bad)
    # without the flag the same calls rebuild the tables and are fine
    again = bwd(other, ws, 0)
    for a_, b_ in zip(again, good):
        assert torch.equal(a_, b_)


def test_pull_prep_buckets_bit_exact():
    """(a2) on the hot path: the (level, image) buckets the prep leaves in the workspace -- bperm / boff, read
    back raw -- against a stable lexsort of the oracle's levels (unique answer -> bit-exact)."""
    wl = inputs.make_workload(5, n_img=5, per_img=333, channels=8)
    cfg = wl.cfg
    rois_np = wl.rois.copy()
    rois_np[7, 0] = -1.0        # invalid batch indices are dropped from the buckets
    rois_np[100, 0] = 2.5
    PH, PW = cfg.out_size
    K, C, L, N = cfg.K, cfg.channels, len(cfg.level_shapes), cfg.n_img
    feats, _ = T.device_feats(wl.feats, "f32", "cl")
    rois = torch.from_numpy(rois_np).cuda()
    out = T.empty_layout((K, C, PH, PW), torch.float32, "cl")
    ws = T.workspace(K, L, PH, PW, 2)
    B.roi_align_fpn_forward(feats, cfg.scales, rois, out, 2, True, cfg.finest_scale, ws)
    torch.cuda.synchronize()
    raw = ws.cpu().numpy()
    align = lambda v: (v + 255) & ~255
    o_bperm = 256
    o_boff = o_bperm + align(4 * K)
    bperm = raw[o_bperm:o_bperm + 4 * K].view(np.int32)
    boff = raw[o_boff:o_boff + 4 * (L * N + 1)].view(np.int32)
    levels = R.assign_levels(rois_np, L, cfg.finest_scale)[0]
    b = rois_np[:, 0]
    valid = (b >= 0) & (b < N) & (b == np.floor(b))
    key = levels.astype(np.int64) * N + np.where(valid, b, 0).astype(np.int64)
    ks = np.nonzero(valid)[0]
    order = ks[np.argsort(key[ks], kind="stable")]
    counts = np.bincount(key[ks], minlength=L * N)
    assert np.array_equal(boff, np.concatenate([[0], np.cumsum(counts)]))
    assert np.array_equal(bperm[:len(order)], order)


def test_forward_ex_no_prep_and_workspace_checks():
    """roi_align_fpn_forward_ex(RAF_NO_PREP): same values, the workspace is neither needed nor touched;
    a misaligned workspace is refused."""
    wl = inputs.make_workload(3, n_img=1, per_img=100, channels=64)
    cfg = wl.cfg
    PH, PW = cfg.out_size
    K, C, L = cfg.K, cfg.channels, len(cfg.level_shapes)
    feats, _ = T.device_feats(wl.feats, "f16", "cl")
    rois = torch.from_numpy(wl.rois).cuda()
    ws = T.workspace(K, L, PH, PW, 2)
    o1 = T.empty_layout((K, C, PH, PW), torch.float16, "cl", fill=float("nan"))
    o2 = T.empty_layout((K, C, PH, PW), torch.float16, "cl", fill=float("nan"))
    B.roi_align_fpn_forward(feats, cfg.scales, rois, o1, 2, True, cfg.finest_scale, ws)
    guard = ws.clone()
    guard.fill_(0x5C)
    B.roi_align_fpn_forward_ex(feats, cfg.scales, rois, o2, 2, True, cfg.finest_scale, B.RAF_NO_PREP, guard)
    B.roi_align_fpn_forward_ex(feats, cfg.scales, rois, o2, 2, True, cfg.finest_scale, B.RAF_NO_PREP, None)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2)
    assert bool((guard == 0x5C).all())
    with pytest.raises(B.RafError) as e:
        B.roi_align_fpn_forward(feats, cfg.scales, rois, o2, 2, True, cfg.finest_scale, ws[16:])
    assert e.value.status == -6


def test_adjoint_identity_on_gpu():
    """<A x, g> = <x, A^T g> with both sides from the CUDA path (fp32): a property at full config-2
    size that needs no oracle."""
    wl = inputs.make_workload(2)
    cfg = wl.cfg
    dev, _ = T.device_feats(wl.feats, "f32", "cl")
    out = T.gpu_forward(dev, cfg.scales, wl.rois, (7, 7), 2, True, 56.0, "cl")
    grads, go = T.gpu_backward(cfg.level_shapes, cfg.scales, wl.grad_out, wl.rois, 2, True, 56.0, "cl")
    lhs = float((out * go).sum())
    rhs = sum(float((g * f.astype(np.float64)).sum()) for g, f in zip(grads, wl.feats))
    scale = float(np.abs(out * go).sum())
    assert abs(lhs - rhs) <= 1e-5 * scale


# ------------------------------------------------------------------------------------------------
# ABI behaviour on the device
# ------------------------------------------------------------------------------------------------
def test_k_zero_and_overwrite_zero_fill():
    shapes = [(1, 8, 10, 12), (1, 8, 5, 6)]
    grads, _ = T.gpu_backward(shapes, [0.25, 0.125], np.zeros((0, 8, 7, 7), np.float32),
                              np.zeros((0, 5), np.float32), 2, True, 56.0, "cl")
    assert all(np.all(g == 0) for g in grads)      # overwrite mode writes every element
    # K == 0 with RAF_REUSE_PREP: the forward wrote nothing into the (garbage-filled) workspace; the
    # backward must not trust it
    grads, _ = T.gpu_backward(shapes, [0.25, 0.125], np.zeros((0, 8, 7, 7), np.float32),
                              np.zeros((0, 5), np.float32), 2, True, 56.0, "cl", flags=B.RAF_REUSE_PREP)
    assert all(np.all(g == 0) for g in grads)


def test_host_entry_points_match_device_path():
    wl = inputs.make_workload(2, n_img=1, per_img=32, channels=32)
    cfg = wl.cfg
    feats_h = [torch.from_numpy(f).permute(0, 2, 3, 1).contiguous().pin_memory().permute(0, 3, 1, 2) for f in wl.feats]
    rois_h = torch.from_numpy(wl.rois).pin_memory()
    out_h = torch.empty((cfg.K, 7, 7, 32), dtype=torch.float32).pin_memory().permute(0, 3, 1, 2)
    nbytes = B.roi_align_fpn_host_arena_bytes(feats_h, cfg.scales, torch.float32, cfg.K, 7, 7, 2)
    arena = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    B.roi_align_fpn_forward_host(feats_h, cfg.scales, rois_h, out_h, 2, True, 56.0, arena)
    torch.cuda.synchronize()
    dev, _ = T.device_feats(wl.feats, "f32", "cl")
    ref = T.gpu_forward(dev, cfg.scales, wl.rois, (7, 7), 2, True, 56.0, "cl")
    assert np.array_equal(out_h.numpy().astype(np.float64), ref)
    gout_h = torch.from_numpy(wl.grad_out).permute(0, 2, 3, 1).contiguous().pin_memory().permute(0, 3, 1, 2)
    grads_h = [torch.empty((s[0], s[2], s[3], s[1]), dtype=torch.float32).pin_memory().permute(0, 3, 1, 2)
               for s in cfg.level_shapes]
    B.roi_align_fpn_backward_host(grads_h, cfg.scales, gout_h, rois_h, 2, True, 56.0, 0, arena)
    torch.cuda.synchronize()
    ref_g, S = R.backward(cfg.level_shapes, cfg.scales, wl.grad_out, wl.rois, (7, 7), 2, True, 56.0)
    T.assert_backward_close([g.numpy().astype(np.float64) for g in grads_h], ref_g, S)


# ------------------------------------------------------------------------------------------------
# guard bands (compute-sanitizer is closed on this GPU pool): every buffer the library writes sits
# inside a larger sentinel-filled allocation; the margins must come back untouched
# ------------------------------------------------------------------------------------------------
def _guarded(nbytes, margin=4096):
    buf = torch.full((nbytes + 2 * margin,), 0x5A, dtype=torch.uint8, device="cuda")
    return buf, buf[margin:margin + nbytes]


def _margins_intact(buf, nbytes, margin=4096):
    return bool((buf[:margin] == 0x5A).all()) and bool((buf[margin + nbytes:] == 0x5A).all())


@pytest.mark.parametrize("index,dtype,kw,P", [
    (2, "f32", dict(n_img=2, per_img=150, channels=64), (7, 7)),
    (5, "bf16", dict(n_img=2, per_img=100, channels=40), (7, 7)),     # boxes partly outside, partial chunk
    (4, "f16", dict(n_img=1, per_img=60, channels=264), (14, 14)),
])
@pytest.mark.parametrize("flags", [0, B.RAF_ATOMIC, B.RAF_REUSE_PREP, B.RAF_PULL_STRIP, B.RAF_PULL_STRIP | B.RAF_REUSE_PREP])
def test_no_out_of_bounds_writes(index, dtype, kw, P, flags):
    wl = inputs.make_workload(index, **kw)
    cfg = wl.cfg
    tdt = T.TORCH_DTYPE[dtype]
    esz = 4 if dtype == "f32" else 2
    K, C, L = cfg.K, cfg.channels, len(cfg.level_shapes)
    PH, PW = P
    feats, _ = T.device_feats(wl.feats, dtype, "cl")
    rois = torch.from_numpy(wl.rois).cuda()
    n_out = K * C * PH * PW
    obuf, oview = _guarded(n_out * esz)
    out = oview.view(tdt).view(K, PH, PW, C).permute(0, 3, 1, 2)
    wsz = B.roi_align_fpn_workspace_bytes(K, L, PH, PW, 2, flags)
    wbuf, ws = _guarded(wsz)
    B.roi_align_fpn_forward(feats, cfg.scales, rois, out, 2, True, cfg.finest_scale, ws)
    gbufs, grads = [], []
    for (n, c, h, w) in cfg.level_shapes:
        gb, gv = _guarded(n * c * h * w * 4)
        gbufs.append((gb, n * c * h * w * 4))
        grads.append(gv.view(torch.float32).view(n, h, w, c).permute(0, 3, 1, 2))
    gout = T.to_layout(torch.randn((K, C, PH, PW), device="cuda").to(tdt), "cl")
    B.roi_align_fpn_backward(grads, cfg.scales, gout, rois, 2, True, cfg.finest_scale, flags, ws)
    torch.cuda.synchronize()
    assert _margins_intact(obuf, n_out * esz), "forward wrote outside its output"
    assert _margins_intact(wbuf, wsz), "workspace overrun"
    for gb, nb in gbufs:
        assert _margins_intact(gb, nb), "backward wrote outside the gradient pyramid"
    assert all(torch.isfinite(g).all() for g in grads) and torch.isfinite(out.float()).all()


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_repack_nchw_forward_and_backward(dtype):
    """RAF_REPACK: dense NCHW operands are repacked to channels-last inside the workspace,
    the channels-last kernels run, the result is repacked back.  Must equal the channels-last call bit for bit
    (same kernels on the same values) and the oracle within tolerance; NaN-filled destinations and a
    garbage-filled workspace; accumulate mode repacks the existing gradients in first."""
    wl = inputs.make_workload(5, n_img=2, per_img=40, channels=32)
    cfg = wl.cfg
    tdt = T.TORCH_DTYPE[dtype]
    PH, PW = cfg.out_size
    K, C, L = cfg.K, cfg.channels, len(cfg.level_shapes)
    rois = torch.from_numpy(wl.rois).cuda()
    f_nchw, exact = T.device_feats(wl.feats, dtype, "nchw")
    f_cl, _ = T.device_feats(wl.feats, dtype, "cl")
    base = B.roi_align_fpn_workspace_bytes(K, L, PH, PW, 2, 0)
    extra = B.roi_align_fpn_repack_bytes(f_nchw, cfg.scales, tdt, K, PH, PW)
    ws = torch.full((base + extra,), 0x7B, dtype=torch.uint8, device="cuda")
    o_nchw = torch.full((K, C, PH, PW), float("nan"), dtype=tdt, device="cuda")
    o_cl = T.empty_layout((K, C, PH, PW), tdt, "cl", fill=float("nan"))
    B.roi_align_fpn_forward_ex(f_nchw, cfg.scales, rois, o_nchw, 2, True, cfg.finest_scale, B.RAF_REPACK, ws)
    B.roi_align_fpn_forward(f_cl, cfg.scales, rois, o_cl, 2, True, cfg.finest_scale, T.workspace(K, L, PH, PW, 2))
    torch.cuda.synchronize()
    assert o_nchw.is_contiguous() and torch.equal(o_nchw, o_cl)
    ref = R.forward(exact, cfg.scales, wl.rois, (PH, PW), 2, True, cfg.finest_scale, coord_f32=True)
    T.assert_forward_close(o_nchw.to(torch.float64).cpu().numpy(), ref, dtype)
    # a workspace without room for the copies is refused; so are operands that are neither layout
    with pytest.raises(B.RafError) as e:
        B.roi_align_fpn_forward_ex(f_nchw, cfg.scales, rois, o_nchw, 2, True, cfg.finest_scale, B.RAF_REPACK, ws[:base])
    assert e.value.status == -6
    with pytest.raises(B.RafError) as e:
        B.roi_align_fpn_forward_ex([f[:, ::2] for f in f_nchw], cfg.scales, rois, o_nchw[:, ::2], 2, True,
                                   cfg.finest_scale, B.RAF_REPACK, ws)
    assert e.value.status == -4
    # backward: overwrite, then accumulate on top of random gradients; RAF_REUSE_PREP works through the repack
    go_t = torch.from_numpy(wl.grad_out).to(tdt)
    go_nchw = go_t.cuda().contiguous()
    go_cl = T.to_layout(go_t.cuda(), "cl")
    rng = np.random.default_rng(5)
    init = [rng.standard_normal(s).astype(np.float32) for s in cfg.level_shapes]
    for flags, start in ((0, None), (B.RAF_ACCUMULATE, init), (B.RAF_REUSE_PREP, None)):
        if start is None:
            g_nchw = [torch.full(s, float("nan"), dtype=torch.float32, device="cuda") for s in cfg.level_shapes]
            g_cl = [T.empty_layout(s, torch.float32, "cl", fill=float("nan")) for s in cfg.level_shapes]
        else:
            g_nchw = [torch.from_numpy(x).cuda().contiguous() for x in start]
            g_cl = [T.to_layout(torch.from_numpy(x).cuda(), "cl") for x in start]
        B.roi_align_fpn_backward(g_nchw, cfg.scales, go_nchw, rois, 2, True, cfg.finest_scale, flags | B.RAF_REPACK, ws)
        B.roi_align_fpn_backward(g_cl, cfg.scales, go_cl, rois, 2, True, cfg.finest_scale, flags & ~B.RAF_REUSE_PREP,
                                 T.workspace(K, L, PH, PW, 2))
        torch.cuda.synchronize()
        for a_, b_ in zip(g_nchw, g_cl):
            assert a_.is_contiguous() and torch.equal(a_, b_)
    gref, S = R.backward(cfg.level_shapes, cfg.scales, go_t.to(torch.float64).numpy(), wl.rois, (PH, PW), 2, True,
                         cfg.finest_scale)
    T.assert_backward_close([t.to(torch.float64).cpu().numpy() for t in g_nchw], gref, S)


@pytest.mark.parametrize("variant", [B.RAF_PULL_TILE, B.RAF_PULL_STRIP])
@pytest.mark.parametrize("index,dtype,kw,P", [
    (4, "bf16", dict(n_img=2, per_img=40, channels=32), None),
    (5, "bf16", dict(n_img=3, per_img=64, channels=64), None),
    (5, "f16", dict(n_img=2, per_img=50, channels=36), None),
    (5, "bf16", dict(n_img=1, per_img=400, channels=16), (7, 7)),     # dense: tiles with several passes / batches
])
def test_backward_16bit_gradient_pyramid(index, dtype, kw, P, variant):
    """roi_align_fpn_backward_ex with the gradient pyramid in grad_out's 16-bit type: fp32 sums
    rounded once per element and pass.  Tolerance: 16-bit rounding of the result (2e-2 relative, north_star's
    figure for 16-bit outputs) + one rounding of a partial sum per extra pass (eps_16 * S, S = sum |terms|)."""
    wl = inputs.make_workload(index, **kw)
    cfg = wl.cfg
    tdt = T.TORCH_DTYPE[dtype]
    PH, PW = P or cfg.out_size
    K, C, L = cfg.K, cfg.channels, len(cfg.level_shapes)
    rng = np.random.default_rng(17)
    gout_np = wl.grad_out if (PH, PW) == tuple(cfg.out_size) else rng.standard_normal((K, C, PH, PW)).astype(np.float32)
    rois = torch.from_numpy(wl.rois).cuda()
    go_t = torch.from_numpy(gout_np).to(tdt)
    go = T.to_layout(go_t.cuda(), "cl")
    ws = T.workspace(K, L, PH, PW, 2)
    gref, S = R.backward(cfg.level_shapes, cfg.scales, go_t.to(torch.float64).numpy(), wl.rois, (PH, PW), 2, True,
                         cfg.finest_scale)
    eps = 2.0 ** -8 if dtype == "bf16" else 2.0 ** -11
    for accumulate in (False, True):
        init = [rng.standard_normal(s).astype(np.float32) for s in cfg.level_shapes]
        if accumulate:
            grads = [T.to_layout(torch.from_numpy(x).to(tdt).cuda(), "cl") for x in init]
            start = [g.to(torch.float64).cpu().numpy() for g in grads]
        else:
            grads = [T.empty_layout(s, tdt, "cl", fill=float("nan")) for s in cfg.level_shapes]
            start = [np.zeros(s) for s in cfg.level_shapes]
        B.roi_align_fpn_backward(grads, cfg.scales, go, rois, 2, True, cfg.finest_scale,
                                 variant | (B.RAF_ACCUMULATE if accumulate else 0), ws)
        torch.cuda.synchronize()
        for g, r, s, st in zip(grads, gref, S, start):
            got = g.to(torch.float64).cpu().numpy()
            want = r + st
            assert np.isfinite(got).all()
            tol = 2e-2 * np.abs(want) + 4 * eps * (s + np.abs(st)) + 1e-6
            assert (np.abs(got - want) <= tol).all(), float((np.abs(got - want) / tol).max())
            if not accumulate:
                assert np.all(got[s == 0] == 0)
    # the combinations the header rules out
    g32 = [T.empty_layout(s, torch.float32, "cl") for s in cfg.level_shapes]
    with pytest.raises(B.RafError) as e:
        B.roi_align_fpn_backward([T.empty_layout(s, tdt, "cl") for s in cfg.level_shapes], cfg.scales, go, rois, 2, True,
                                 cfg.finest_scale, B.RAF_ATOMIC, ws)
    assert e.value.status == -5
    with pytest.raises(ValueError):
        B.roi_align_fpn_backward([t.to(torch.float64) for t in g32], cfg.scales, go, rois, 2, True, cfg.finest_scale, 0, ws)
