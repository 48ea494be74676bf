"""The C-ABI library loads and exports every symbol include/raf.h declares; host-detectable argument
errors are reported as negative raf_status without touching the device (no compute call here)."""
import ctypes
import os
import re

import pytest

from paper_1906_07155_b200 import binding as B
from paper_1906_07155_b200 import build as raf_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    raf_build.build()
    return B.lib()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "raf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(roi_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert len(names) >= 9
    assert set(names) == set(B.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None


def test_no_torch_types_in_header():
    src = open(os.path.join(ROOT, "include", "raf.h")).read()
    assert "torch" not in src and "at::" not in src and "#include <cuda" not in src


def test_strerror(lib):
    assert B.strerror(0) == "ok"
    for code in range(-7, 0):
        assert B.strerror(code) not in ("ok", "unknown status")
    assert B.strerror(-99) == "unknown status"


def test_workspace_bytes_monotone(lib):
    a = B.roi_align_fpn_workspace_bytes(0, 4, 7, 7, 2)
    b = B.roi_align_fpn_workspace_bytes(1024, 4, 7, 7, 2)
    c = B.roi_align_fpn_workspace_bytes(8192, 4, 7, 7, 2, B.RAF_DETERMINISTIC)
    assert 0 < a <= b <= c and a % 256 == 0 and b % 256 == 0 and c % 256 == 0


def _levels(L=2, data=0x1000, **over):
    """Two consistent levels; keyword overrides apply to the LAST level only."""
    n, c, h, w = 1, 8, 10, 12
    arr = (B.RafLevel * L)()
    for i in range(L):
        arr[i].data = data
        arr[i].n, arr[i].c, arr[i].h, arr[i].w = n, c, h, w
        arr[i].sn, arr[i].sc, arr[i].sh, arr[i].sw = c * h * w, 1, w * c, c
        arr[i].spatial_scale = 0.25 / (1 << i)
    for k, v in over.items():
        setattr(arr[L - 1], k, v)
    return arr


def _fwd(lib, lv, L=2, dtype=0, rois=0x2000, K=4, ph=7, pw=7, g=2, out=0x3000, strides=(392, 1, 56, 8),
         ws=0x4000, ws_bytes=1 << 20, fs=56.0):
    st = (ctypes.c_int64 * 4)(*strides) if strides is not None else None
    return lib.roi_align_fpn_forward(lv, L, dtype, rois, K, ph, pw, g, 1, fs, out, st, ws, ws_bytes, None)


def test_forward_argument_errors(lib):
    assert _fwd(lib, None) == -1                                   # RAF_ERR_NULL
    assert _fwd(lib, _levels(), rois=None) == -1
    assert _fwd(lib, _levels(), out=None) == -1
    assert _fwd(lib, _levels(), ws=None) == -1
    assert _fwd(lib, _levels(), strides=None) == -1
    assert _fwd(lib, _levels(data=None)) == -1
    assert _fwd(lib, _levels(), L=0) == -2                         # RAF_ERR_SHAPE
    assert _fwd(lib, _levels(), L=9) == -2
    assert _fwd(lib, _levels(), K=-1) == -2
    assert _fwd(lib, _levels(), ph=0) == -2
    assert _fwd(lib, _levels(), pw=33) == -2
    assert _fwd(lib, _levels(), g=-1) == -2
    assert _fwd(lib, _levels(c=4)) == -2                           # c mismatch across levels
    assert _fwd(lib, _levels(n=3)) == -2
    assert _fwd(lib, _levels(h=0)) == -2
    assert _fwd(lib, _levels(), fs=0.0) == -2
    assert _fwd(lib, _levels(), dtype=7) == -3                     # RAF_ERR_DTYPE
    assert _fwd(lib, _levels(sw=0)) == -4                          # RAF_ERR_STRIDE
    assert _fwd(lib, _levels(), strides=(392, 1, 0, 8)) == -4
    assert _fwd(lib, _levels(), ws_bytes=8) == -6                  # RAF_ERR_WORKSPACE
    assert _fwd(lib, _levels(), K=0, rois=None, out=None, ws=None) == 0   # K == 0: nothing to do


def test_backward_argument_errors(lib):
    st = (ctypes.c_int64 * 4)(392, 1, 56, 8)

    def bwd(lv, L=2, dtype=0, gout=0x3000, strides=st, rois=0x2000, K=4, flags=0, ws=0x4000, ws_bytes=1 << 20):
        return lib.roi_align_fpn_backward(lv, L, dtype, gout, strides, rois, K, 7, 7, 2, 1, 56.0, flags, ws,
                                          ws_bytes, None)
    assert bwd(None) == -1
    assert bwd(_levels(), gout=None) == -1
    assert bwd(_levels(), rois=None) == -1
    assert bwd(_levels(), strides=None) == -1
    assert bwd(_levels(), K=-2) == -2
    assert bwd(_levels(), dtype=3) == -3
    assert bwd(_levels(sn=-5)) == -4
    assert bwd(_levels(), flags=1024) == -5                        # RAF_ERR_UNSUPPORTED (unknown flag)
    assert bwd(_levels(), flags=32 | 64) == -5                     # RAF_PULL_STRIP with RAF_PULL_TILE
    assert bwd(_levels(), ws_bytes=0) == -6


def test_assign_levels_argument_errors(lib):
    f = lib.roi_fpn_assign_levels
    assert f(None, 4, 4, 56.0, None, None, None, None, 0, None) == -1
    assert f(0x1000, -1, 4, 56.0, None, None, None, None, 0, None) == -2
    assert f(0x1000, 4, 0, 56.0, None, None, None, None, 0, None) == -2
    assert f(0x1000, 4, 9, 56.0, None, None, None, None, 0, None) == -2
    assert f(0x1000, 4, 4, -1.0, None, None, None, None, 0, None) == -2
    assert f(None, 0, 4, 56.0, None, None, None, None, 0, None) == 0


def test_product_does_not_import_oracle():
    """The product package never routes through the oracle or any CPU fallback."""
    pkg = os.path.join(ROOT, "paper_1906_07155_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), fn
                assert "raf_ref" not in text and "oracle/" not in text, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".cpp")):
            text = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "import paper_1906_07155_b200" not in text and "from paper_1906_07155_b200" not in text
            assert "libraf.so" not in text and "binding" not in text


def test_binding_rejects_what_the_abi_cannot_see():
    """binding.py validates dtypes / shapes / contiguity / devices before the raw pointers go down
    (ValueError, no library call): the C ABI cannot see any of it."""
    import torch
    feats = [torch.zeros((1, 4, 8, 8)), torch.zeros((1, 4, 4, 4))]
    rois = torch.zeros((3, 5))
    out = torch.zeros((3, 4, 7, 7))
    ws = torch.zeros(1024, dtype=torch.uint8)
    scales = [0.25, 0.125]
    call = lambda **kw: B.roi_align_fpn_forward(kw.get("feats", feats), scales, kw.get("rois", rois), kw.get("out", out),
                                                2, True, 56.0, ws)
    bad = [dict(rois=rois.double()), dict(rois=torch.zeros((3, 6))), dict(rois=torch.zeros((5, 3)).t()),
           dict(rois=torch.zeros((4, 5))),                      # K differs from out
           dict(out=torch.zeros((3, 8, 7, 7))),                 # C differs from the levels
           dict(out=out.half()),                                # dtype differs from the features
           dict(feats=[feats[0], torch.zeros((1, 8, 4, 4))]),   # C differs across levels
           dict(feats=[feats[0], feats[1].half()]),
           dict()]                                              # all valid but on the CPU: not CUDA tensors
    for kw in bad:
        with pytest.raises(ValueError):
            call(**kw)
    grads = [torch.zeros((1, 4, 8, 8)), torch.zeros((1, 4, 4, 4), dtype=torch.bfloat16)]
    with pytest.raises(ValueError):   # gradient pyramid must be fp32
        B.roi_align_fpn_backward(grads, scales, out, rois, 2, True, 56.0, 0, ws)


def _levels_nchw(L=2, n=2, c=8, h=16, w=20):
    arr = (B.RafLevel * L)()
    for i in range(L):
        hh, ww = max(h >> i, 1), max(w >> i, 1)
        arr[i].data = 0x100000 * (i + 1)
        arr[i].n, arr[i].c, arr[i].h, arr[i].w = n, c, hh, ww
        arr[i].sn, arr[i].sc, arr[i].sh, arr[i].sw = c * hh * ww, hh * ww, ww, 1
        arr[i].spatial_scale = 0.25 / (1 << i)
    return arr


def _levels_c(c, L=2):
    arr = _levels(L)
    for i in range(L):
        arr[i].c = c
        arr[i].sn, arr[i].sh, arr[i].sw = c * arr[i].h * arr[i].w, arr[i].w * c, c
    return arr


def test_round2_entry_points_reject_bad_arguments_before_any_launch(lib):
    """Host-side validation of the entry points added in round 2 (fake pointers: nothing may be launched)."""
    i64x4 = ctypes.c_int64 * 4
    cl, nchw = i64x4(392, 1, 56, 8), i64x4(392, 49, 7, 1)
    f = ctypes.c_float
    # backward_ex: the gradient pyramid is fp32 or has the 16-bit type of grad_out
    bex = lambda gdt, odt, flags=0: lib.roi_align_fpn_backward_ex(_levels(), 2, odt, gdt, 0x3000, cl, 0x2000, 4, 7, 7, 2, 1,
                                                                  f(56.0), flags, 0x4000, 1 << 20, None)
    assert bex(1, 2) == -5 and bex(2, 0) == -5 and bex(7, 0) == -3
    assert bex(2, 2, flags=4) == -5 and bex(2, 2, flags=128) == -5      # RAF_ATOMIC / RAF_REPACK with a 16-bit pyramid
    # RAF_REPACK: needs dense NCHW operands and room for the copies
    lib.roi_align_fpn_repack_bytes.restype = ctypes.c_size_t
    lib.roi_align_fpn_workspace_bytes.restype = ctypes.c_size_t
    need = lib.roi_align_fpn_repack_bytes(_levels_nchw(), 2, 0, 4, 7, 7)
    assert need >= 4 * (2 * 8 * 16 * 20 + 2 * 8 * 8 * 10) + 4 * 4 * 8 * 49 and need % 256 == 0
    assert lib.roi_align_fpn_repack_bytes(None, 2, 0, 4, 7, 7) == 0
    fex = lambda lv, st, ws_bytes: lib.roi_align_fpn_forward_ex(lv, 2, 0, 0x2000, 4, 7, 7, 2, 1, f(56.0), 0x3000, st, 128, 0x4000,
                                                                ws_bytes, None)
    base = lib.roi_align_fpn_workspace_bytes(4, 2, 7, 7, 2, 0)
    assert fex(_levels_nchw(), nchw, base + need - 1) == -6
    assert fex(_levels_nchw(), i64x4(392, 49, 14, 1), 1 << 24) == -4       # output neither channels-last nor dense NCHW
    # fused gather + FC
    fc = lambda dtype=2, g=2, n_out=512, lv=None: lib.roi_align_fc_fpn_forward(lv or _levels_c(64), 2, dtype, 0x2000, 4, 7, 7, g, 1,
                                                                                f(56.0), 0x5000, None, n_out, 0x6000, None)
    assert fc(dtype=0) == -5 and fc(g=3) == -5 and fc(n_out=256) == -5 and fc(lv=_levels()) == -5 and fc(n_out=0) == -2
    assert lib.roi_align_fc_fpn_forward(_levels_c(64), 2, 2, 0x2000, 4, 7, 7, 2, 1, f(56.0), None, None, 512, 0x6000, None) == -1
    # deformable RoI pooling
    dfw = lambda g=2, out=0x3000: lib.roi_deform_pool_fpn_forward(_levels(), 2, 0, 0x2000, 4, None, f(0.1), 7, 7, g, f(56.0), out, cl, None)
    assert dfw(g=-1) == -2 and dfw(out=None) == -1
    assert lib.roi_deform_pool_fpn_backward(_levels(), None, 2, 0, 0x3000, cl, 0x2000, 4, None, f(0.1), 7, 7, 2, f(56.0), None, 4,
                                            None) == -5
    assert lib.roi_deform_pool_fpn_backward(_levels(), _levels(h=9), 2, 0, 0x3000, cl, 0x2000, 4, None, f(0.1), 7, 7, 2, f(56.0),
                                            None, 0, None) == -2
