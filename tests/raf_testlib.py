"""Helpers for the GPU parity tests: device tensors in a given physical layout, calls through the
C ABI binding, and the tolerance forms of DESIGN.md section 3 (readings S10, S11)."""
import numpy as np
import torch

from paper_1906_07155_b200 import binding as B

TORCH_DTYPE = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}


def to_layout(x_nchw: torch.Tensor, layout: str) -> torch.Tensor:
    """Return a logical-[N,C,H,W] tensor whose physical order is NCHW ('nchw') or NHWC ('cl')."""
    if layout == "nchw":
        return x_nchw.contiguous()
    assert layout == "cl"
    return x_nchw.permute(0, 2, 3, 1).contiguous().permute(0, 3, 1, 2)


def empty_layout(shape, dtype, layout: str, device="cuda", fill=None) -> torch.Tensor:
    n, c, h, w = shape
    if layout == "nchw":
        t = torch.empty((n, c, h, w), dtype=dtype, device=device)
    else:
        t = torch.empty((n, h, w, c), dtype=dtype, device=device).permute(0, 3, 1, 2)
    if fill is not None:
        t.fill_(fill)
    return t


def workspace(K, L, PH, PW, g, flags=0):
    """Workspace filled with a non-zero pattern: stale contents must never be trusted by the library."""
    return torch.full((B.roi_align_fpn_workspace_bytes(K, L, PH, PW, g, flags),), 0x7B, dtype=torch.uint8, device="cuda")


def device_feats(feats_np, dtype: str, layout: str):
    """fp32 numpy [N,C,H,W] -> device tensors of `dtype` in `layout`; also returns the exact float64
    widening of what the device holds (the oracle's input)."""
    dev, exact = [], []
    for f in feats_np:
        t = torch.from_numpy(f).to(TORCH_DTYPE[dtype])
        exact.append(t.to(torch.float64).numpy())
        dev.append(to_layout(t.cuda(), layout))
    return dev, exact


def gpu_forward(feats_dev, scales, rois_np, out_size, g, aligned, finest_scale, layout):
    K = rois_np.shape[0]
    C = feats_dev[0].shape[1]
    PH, PW = out_size
    rois = torch.from_numpy(np.ascontiguousarray(rois_np, np.float32)).cuda()
    out = empty_layout((K, C, PH, PW), feats_dev[0].dtype, layout, fill=float("nan"))
    ws = workspace(K, len(feats_dev), PH, PW, g)
    B.roi_align_fpn_forward(feats_dev, scales, rois, out, g, aligned, finest_scale, ws)
    torch.cuda.synchronize()
    return out.to(torch.float64).cpu().numpy()


def gpu_backward(shapes, scales, gout_np, rois_np, g, aligned, finest_scale, layout, gout_dtype="f32",
                 flags=0, init=None):
    """Returns (grads list of float64 numpy in logical NCHW, exact float64 gout the device saw)."""
    K = rois_np.shape[0]
    rois = torch.from_numpy(np.ascontiguousarray(rois_np, np.float32)).cuda()
    go_t = torch.from_numpy(np.ascontiguousarray(gout_np, np.float32)).to(TORCH_DTYPE[gout_dtype])
    go_exact = go_t.to(torch.float64).numpy()
    go = to_layout(go_t.cuda(), layout)
    grads = []
    for i, s in enumerate(shapes):
        if init is not None:
            grads.append(to_layout(torch.from_numpy(init[i]).float().cuda(), layout))
        else:
            grads.append(empty_layout(s, torch.float32, layout, fill=float("nan")))
    PH, PW = gout_np.shape[2:]
    ws = workspace(K, len(shapes), PH, PW, g, flags)
    B.roi_align_fpn_backward(grads, scales, go, rois, g, aligned, finest_scale, flags, ws)
    torch.cuda.synchronize()
    return [t.to(torch.float64).cpu().numpy() for t in grads], go_exact


def assert_forward_close(gpu, ref, dtype: str):
    """Reading S10: |gpu-ref| <= 1e-6 + 1e-5|ref| (fp32);  <= 1e-6 + 2e-2|ref| (fp16/bf16 in/out,
    fp32 accumulate; ref = double result before rounding)."""
    rtol = 1e-5 if dtype == "f32" else 2e-2
    err = np.abs(gpu - ref)
    tol = 1e-6 + rtol * np.abs(ref)
    bad = err > tol
    assert not bad.any(), (f"{int(bad.sum())} of {bad.size} outside tolerance; worst err/tol = "
                           f"{float((err / tol).max()):.3f} at {np.unravel_index(np.argmax(err / tol), err.shape)}")
    return float((err / tol).max())


def assert_backward_close(gpu, ref, S):
    """Reading S11: |gpu-ref| <= 1e-4|ref| + 1e-6*S, S = sum |w*gout/count| per element; plus the
    norm-wise form max|d| / max|ref| <= 1e-4.  Elements nothing scatters to must be exactly 0."""
    worst = 0.0
    for g, r, s in zip(gpu, ref, S):
        assert np.isfinite(g).all()
        err = np.abs(g - r)
        tol = 1e-4 * np.abs(r) + 1e-6 * s
        bad = err > tol
        assert not bad.any(), f"{int(bad.sum())} of {bad.size} outside tolerance"
        assert np.all(g[s == 0] == 0)
        if np.abs(r).max() > 0:
            assert err.max() / np.abs(r).max() <= 1e-4
        with np.errstate(invalid="ignore", divide="ignore"):
            q = np.where(tol > 0, err / tol, 0.0)
        worst = max(worst, float(q.max()))
    return worst
