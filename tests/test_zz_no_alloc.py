"""roi_align_fpn_backward_static (include/raf.h): the backward for callers that cannot allocate -- its scratch is a
static device array inside the library.  The GPU test compares it with the existing path (roi_align_fpn_backward with a
caller workspace) on calls made one after the other; the host tests check the size limit and the refused flags.

Collected last on purpose (the suite runs with `pytest -x`): a failure here must not hide any other test."""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

from oracle import raf_ref as R
from paper_1906_07155_b200 import binding as B
from paper_1906_07155_b200 import build as raf_build
from paper_1906_07155_b200 import inputs
import raf_testlib as T

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _fake_levels(L=2):
    n, c, h, w = 1, 8, 10, 12
    arr = (B.RafLevel * L)()
    for i in range(L):
        arr[i].data = 0x1000
        arr[i].n, arr[i].c, arr[i].h, arr[i].w = n, c, h, w
        arr[i].sn, arr[i].sc, arr[i].sh, arr[i].sw = c * h * w, 1, w * c, c
        arr[i].spatial_scale = 0.25 / (1 << i)
    return arr


def test_static_entry_point_limit_and_flags_decided_on_the_host():
    """No GPU needed: the size limit and the refused flags are decided before any CUDA call."""
    raf_build.build()
    lib = B.lib()
    st = (ctypes.c_int64 * 4)(392, 1, 56, 8)

    def call(K=4, ph=7, pw=7, g=2, flags=0):
        return lib.roi_align_fpn_backward_static(_fake_levels(), 2, 0, 0x3000, st, 0x2000, K, ph, pw, g, 1, 56.0, flags, None)
    assert B.RAF_STATIC_WS_BYTES == 4 << 20
    # the stated capacity: 8192 RoIs at 7 x 7 bins and 4096 at 14 x 14 fit, more does not
    assert B.roi_align_fpn_workspace_bytes(8192, 4, 7, 7, 2, 0) <= B.RAF_STATIC_WS_BYTES
    assert B.roi_align_fpn_workspace_bytes(4096, 4, 14, 14, 2, 0) <= B.RAF_STATIC_WS_BYTES
    assert B.roi_align_fpn_workspace_bytes(16384, 4, 7, 7, 2, 0) > B.RAF_STATIC_WS_BYTES
    assert call(K=16384) == -6                       # RAF_ERR_WORKSPACE: beyond the static array
    assert call(K=8192, ph=14, pw=14) == -6
    assert call(K=200000, ph=32, pw=32, g=8) == -6
    assert call(flags=B.RAF_REUSE_PREP) == -5        # RAF_ERR_UNSUPPORTED
    assert call(flags=B.RAF_REPACK) == -5
    assert "workspace" in B.strerror(-6)


def test_static_entry_point_source_allocates_nothing():
    src = open(os.path.join(ROOT, "paper_1906_07155_b200", "csrc", "raf_static.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)
    assert not re.search(r"cudaMalloc|cudaFree|cudaHostAlloc|cublas|new\s|malloc\s*\(", code)
    assert "cudaGetSymbolAddress" in code and "__align__(256)" in code


def _case(wl, dtype, flags, P=None, g=None):
    """One backward through the existing path (caller workspace) and one through the static entry point, same inputs."""
    cfg = wl.cfg
    P = tuple(P or cfg.out_size)
    g = cfg.sampling_ratio if g is None else g
    gout = wl.grad_out
    if gout.shape[2:] != P:
        gout = np.random.default_rng(5).standard_normal((cfg.K, cfg.channels, *P)).astype(np.float32)
    rois = torch.from_numpy(np.ascontiguousarray(wl.rois, np.float32)).cuda()
    go_t = torch.from_numpy(np.ascontiguousarray(gout, np.float32)).to(T.TORCH_DTYPE[dtype])
    go_exact = go_t.to(torch.float64).numpy()
    go = T.to_layout(go_t.cuda(), "cl")
    K, L = cfg.K, len(cfg.level_shapes)

    old = [T.empty_layout(s, torch.float32, "cl", fill=float("nan")) for s in cfg.level_shapes]
    ws = T.workspace(K, L, P[0], P[1], g, flags)
    B.roi_align_fpn_backward(old, cfg.scales, go, rois, g, cfg.aligned, cfg.finest_scale, flags, ws)
    new = [T.empty_layout(s, torch.float32, "cl", fill=float("nan")) for s in cfg.level_shapes]
    B.roi_align_fpn_backward_static(new, cfg.scales, go, rois, g, cfg.aligned, cfg.finest_scale, flags)
    torch.cuda.synchronize()

    old_np = [t.to(torch.float64).cpu().numpy() for t in old]
    new_np = [t.to(torch.float64).cpu().numpy() for t in new]
    ref, S = R.backward(cfg.level_shapes, cfg.scales, go_exact, wl.rois, P, g, cfg.aligned, cfg.finest_scale, coord_f32=True)
    T.assert_backward_close(new_np, old_np, S)   # against the existing path, tolerance of reading S11
    T.assert_backward_close(new_np, ref, S)      # and against the oracle
    return new_np, old_np


@pytest.mark.gpu
def test_static_entry_point_matches_the_existing_path_on_calls_in_a_row():
    # four calls in a row on the one shared array, with different table sizes and contents in between: a larger fp32
    # batch, a smaller bf16 batch with 14 x 14 bins (the array still holds the first call's longer tables), the
    # atomic variant, and the first again
    a = inputs.make_workload(2, n_img=2, per_img=96, channels=64)
    b = inputs.make_workload(4, n_img=2, per_img=40, channels=32)
    first, first_old = _case(a, "f32", B.RAF_DETERMINISTIC)
    _case(b, "bf16", 0)
    _case(b, "bf16", B.RAF_PULL_STRIP)
    _case(a, "f32", B.RAF_ATOMIC)
    again, _ = _case(a, "f32", B.RAF_DETERMINISTIC)
    for x, y, z in zip(first, again, first_old):   # deterministic kernels: the same bits every time, on both paths
        assert np.array_equal(x, y)
        assert np.array_equal(x, z)


@pytest.mark.gpu
def test_static_entry_point_accumulates_and_takes_empty_batches():
    wl = inputs.make_workload(1)
    cfg = wl.cfg
    rois = torch.from_numpy(np.ascontiguousarray(wl.rois, np.float32)).cuda()
    go = T.to_layout(torch.from_numpy(wl.grad_out).cuda(), "cl")
    g = cfg.sampling_ratio
    new = [T.empty_layout(s, torch.float32, "cl", fill=0.0) for s in cfg.level_shapes]
    B.roi_align_fpn_backward_static(new, cfg.scales, go, rois, g, cfg.aligned, cfg.finest_scale, 0)
    once = [t.clone() for t in new]
    B.roi_align_fpn_backward_static(new, cfg.scales, go, rois, g, cfg.aligned, cfg.finest_scale, B.RAF_ACCUMULATE)
    torch.cuda.synchronize()
    for t, o in zip(new, once):
        assert torch.allclose(t, 2 * o, rtol=1e-5, atol=1e-6)
    # K = 0: every gradient element is written (zero)
    empty = [T.empty_layout(s, torch.float32, "cl", fill=float("nan")) for s in cfg.level_shapes]
    B.roi_align_fpn_backward_static(empty, cfg.scales, go[:0], rois[:0], g, cfg.aligned, cfg.finest_scale, 0)
    torch.cuda.synchronize()
    for t in empty:
        assert torch.count_nonzero(t).item() == 0
