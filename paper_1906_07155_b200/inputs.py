"""Seeded synthetic workloads (numpy only) shared by the oracle-side tests, the CUDA-side tests and
bench.py.  Holds NONE of the method's arithmetic: it only draws boxes, features and gradients.

The paper's workloads are COCO 2017 images resized to 1333x800, 2 images per GPU (PAPER.md:142-144,
section 4.1); COCO, trained weights and real proposals are not available, so these inputs take
their shapes, counts and size distributions from BASELINE.json `configs` and stand in for them
(recipe: SURVEY.md 8(d), restated in DESIGN.md section 4).
"""
import math
from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

SEED_BASE = 190607155
IMG_H, IMG_W = 800, 1344
FPN_STRIDES = (4, 8, 16, 32)


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config."""
    index: int
    name: str
    n_img: int
    per_img: int
    dtype: str                      # "f32" | "f16" | "bf16"
    out_size: Tuple[int, int]
    side_lo: float = 16.0
    side_hi: float = 800.0
    clip: bool = True               # reading S15
    backward: bool = True
    channels: int = 256
    sampling_ratio: int = 2
    aligned: bool = True            # reading S14
    finest_scale: float = 56.0      # reading S14
    strides: Tuple[int, ...] = FPN_STRIDES
    img_hw: Tuple[int, int] = (IMG_H, IMG_W)
    level_hist: Optional[Tuple[int, ...]] = None   # SURVEY 8(d) reproducibility pin

    @property
    def K(self) -> int:
        return self.n_img * self.per_img

    @property
    def level_shapes(self) -> List[Tuple[int, int, int, int]]:
        if self.index == 1:
            return [(1, self.channels, 16, 16)]
        H, W = self.img_hw
        return [(self.n_img, self.channels, H // s, W // s) for s in self.strides]

    @property
    def scales(self) -> List[float]:
        if self.index == 1:
            return [1.0]
        return [1.0 / s for s in self.strides]


CONFIGS = {
    1: Config(1, "tiny single-level", 1, 8, "f32", (7, 7), channels=4, strides=(1,),
              img_hw=(16, 16), level_hist=(8,)),
    2: Config(2, "Faster R-CNN R-50-FPN box head (training)", 2, 512, "f32", (7, 7),
              level_hist=(534, 176, 204, 110)),
    3: Config(3, "Faster R-CNN inference", 1, 1000, "f16", (7, 7), backward=False,
              level_hist=(512, 188, 190, 110)),
    4: Config(4, "Mask R-CNN mask head", 2, 128, "bf16", (14, 14), side_lo=32.0, side_hi=600.0,
              level_hist=(122, 70, 53, 11)),
    5: Config(5, "large-batch mixed precision", 16, 512, "bf16", (7, 7), side_lo=8.0,
              side_hi=1000.0, clip=False, level_hist=(4473, 1208, 1151, 1360)),
}


def make_rois(cfg: Config, rng: np.random.Generator) -> np.ndarray:
    """rois[K,5] = (batch_idx, x1, y1, x2, y2) in image pixels, fp32."""
    K = cfg.K
    if cfg.index == 1:
        xs = np.sort(rng.uniform(0, 16, (K, 2)), axis=1)
        ys = np.sort(rng.uniform(0, 16, (K, 2)), axis=1)
        return np.stack([np.zeros(K), xs[:, 0], ys[:, 0], xs[:, 1], ys[:, 1]], 1).astype(np.float32)
    H, W = cfg.img_hw
    side = np.exp(rng.uniform(math.log(cfg.side_lo), math.log(cfg.side_hi), K))
    asp = np.exp(rng.uniform(math.log(0.5), math.log(2.0), K))
    cx = rng.uniform(0, W, K)
    cy = rng.uniform(0, H, K)
    w = side * np.sqrt(asp)
    h = side / np.sqrt(asp)
    x1, y1, x2, y2 = cx - w / 2, cy - h / 2, cx + w / 2, cy + h / 2
    if cfg.clip:
        x1, x2 = np.clip(x1, 0, W), np.clip(x2, 0, W)
        y1, y2 = np.clip(y1, 0, H), np.clip(y2, 0, H)
    b = (np.arange(K) // cfg.per_img).astype(np.float64)
    return np.stack([b, x1, y1, x2, y2], 1).astype(np.float32)


@dataclass
class Workload:
    cfg: Config
    rois: np.ndarray                       # [K,5] fp32
    feats: List[np.ndarray] = field(default_factory=list)   # per level, logical NCHW fp32
    grad_out: Optional[np.ndarray] = None  # [K,C,PH,PW] fp32


def make_workload(index: int, with_feats: bool = True, with_grad: bool = True,
                  n_img: Optional[int] = None, per_img: Optional[int] = None,
                  channels: Optional[int] = None) -> Workload:
    """Draw order (fixed): RoI vectors, then features per level (logical NCHW, fp32 standard normal),
    then grad_out.  n_img / per_img / channels override the config for reduced-size parity cases
    (the stream then differs from the full config's; histogram pins apply to the full size only)."""
    cfg = CONFIGS[index]
    if n_img is not None or per_img is not None or channels is not None:
        cfg = Config(**{**cfg.__dict__, "n_img": n_img or cfg.n_img, "per_img": per_img or cfg.per_img,
                        "channels": channels or cfg.channels, "level_hist": None})
    rng = np.random.default_rng(SEED_BASE + index)
    rois = make_rois(cfg, rng)
    wl = Workload(cfg, rois)
    if with_feats:
        wl.feats = [rng.standard_normal(s, dtype=np.float32) for s in cfg.level_shapes]
    if with_grad:
        if not with_feats:  # keep the stream position independent of with_feats
            for s in cfg.level_shapes:
                rng.standard_normal(s, dtype=np.float32)
        PH, PW = cfg.out_size
        wl.grad_out = rng.standard_normal((cfg.K, cfg.channels, PH, PW), dtype=np.float32)
    return wl


def adversarial_level_rois(finest_scale: float = 56.0, L: int = 4, ulps: int = 16) -> np.ndarray:
    """Square boxes whose side sweeps +-`ulps` fp32 steps around every level boundary, plus
    degenerate boxes (zero / negative extent).  Pure input construction: no level is computed."""
    rows = []
    for j in range(1, L + 1):
        centre = np.float32(finest_scale * 2.0 ** j)
        s = centre
        for _ in range(ulps):
            s = np.nextafter(s, np.float32(0))
        for _ in range(2 * ulps + 1):
            rows.append((0.0, 10.0, 20.0, 10.0 + float(s), 20.0 + float(s)))
            rows.append((0.0, 0.0, 0.0, float(s), float(s)))
            s = np.nextafter(s, np.float32(np.inf))
    rows += [(0, 5, 5, 5, 50), (0, 5, 5, 50, 5), (0, 50, 5, 5, 50), (0, 50, 50, 5, 5),
             (0, 0, 0, 0, 0), (0, 0, 0, 1e-3, 1e-3), (0, -100, -100, 3000, 3000)]
    return np.asarray(rows, dtype=np.float32)
