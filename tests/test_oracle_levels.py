"""Pins for the oracle's level assignment and bucketing (readings S2-S4).

None of these re-types the oracle's comparison chain: they use worked values, an exact-arithmetic
evaluation (Python integers / Fraction on the fp32 bit patterns), a float64 evaluation with the
allowed-disagreement band, seeded histograms from the survey probe, and numpy's stable argsort.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from conftest import read_golden
from oracle import raf_ref as R
from paper_1906_07155_b200 import inputs


def sq(side, x0=0.0, y0=0.0):
    return [0.0, x0, y0, x0 + side, y0 + side]


def levels_of(rows, L=4, fs=56.0):
    return R.assign_levels(np.asarray(rows, np.float32), L, fs)[0].tolist()


def test_worked_values():
    # SURVEY 8(c) pin row "level map": exact in real arithmetic
    assert levels_of([sq(112.0)]) == [1]
    assert levels_of([sq(224.0)]) == [2]
    assert levels_of([sq(448.0)]) == [3]
    assert levels_of([sq(896.0)]) == [3]       # clamps to L-1
    assert levels_of([sq(3000.0)]) == [3]
    assert levels_of([sq(56.0)]) == [0]
    assert levels_of([sq(1.0)]) == [0]
    # smallest square side reaching level 1 is about 56*(2 - 1e-6) = 111.999944
    assert levels_of([sq(np.float32(111.99995))]) == [1]
    assert levels_of([sq(np.float32(111.99994))]) == [0]
    # degenerate boxes: w*h == 0 and w*h < 0 (sqrt -> NaN) -> level 0 (reading S4)
    assert levels_of([[0, 5, 5, 5, 50], [0, 5, 5, 50, 5], [0, 50, 5, 5, 50], [0, 0, 0, 0, 0]]) == [0, 0, 0, 0]
    # both extents negative: product positive -> a normal level (formula applied literally, S8)
    assert levels_of([[0, 300, 300, 76, 76]]) == [2]
    # fewer levels clamp lower
    assert levels_of([sq(448.0)], L=2) == [1]
    assert levels_of([sq(448.0)], L=1) == [0]


def _exact_level(roi, L, fs):
    """Independent evaluation: every fp32 step done by numpy's correctly rounded float32 scalar ops,
    and the final floor(log2 t) taken EXACTLY from the binary exponent of t (math.frexp)."""
    f = np.float32
    w = f(roi[3]) - f(roi[1])
    h = f(roi[4]) - f(roi[2])
    with np.errstate(invalid="ignore"):
        t = f(np.sqrt(f(w * h))) / f(fs) + f(1e-6)
    if not np.isfinite(t):
        return L - 1 if t > 0 else 0
    if t <= 0:
        return 0
    m, e = math.frexp(float(t))      # t = m * 2^e, 0.5 <= m < 1  -> floor(log2 t) = e - 1
    return int(min(max(e - 1, 0), L - 1))


def test_boundary_sweep_exact_exponent():
    rois = inputs.adversarial_level_rois()
    got = R.assign_levels(rois, 4, 56.0)[0]
    exp = np.array([_exact_level(r, 4, 56.0) for r in rois])
    assert np.array_equal(got, exp)
    # the sweep really straddles every boundary
    assert set(got.tolist()) == {0, 1, 2, 3}


def test_float64_evaluation_disagrees_only_near_boundaries():
    rng = np.random.default_rng(7)
    K = 20000
    side = np.exp(rng.uniform(math.log(4), math.log(2000), K))
    asp = np.exp(rng.uniform(math.log(0.25), math.log(4), K))
    w, h = side * np.sqrt(asp), side / np.sqrt(asp)
    x1, y1 = rng.uniform(0, 1000, K), rng.uniform(0, 1000, K)
    rois = np.stack([np.zeros(K), x1, y1, x1 + w, y1 + h], 1).astype(np.float32)
    got = R.assign_levels(rois, 4, 56.0)[0]
    r64 = rois.astype(np.float64)
    t = np.sqrt((r64[:, 3] - r64[:, 1]) * (r64[:, 4] - r64[:, 2])) / 56.0 + 1e-6
    ref = np.clip(np.floor(np.log2(t)), 0, 3).astype(np.int32)
    bad = got != ref
    # disagreement allowed only within 4 fp32 ulp of a power of two (SURVEY 8(c) pin row)
    near = np.zeros(K, bool)
    for j in (1, 2, 3):
        near |= np.abs(t - 2.0 ** j) <= 4 * np.spacing(np.float32(2.0 ** j))
    assert not np.any(bad & ~near)
    assert bad.sum() < 10


def test_seeded_histograms(golden_dir):
    gold = read_golden(os.path.join(golden_dir, "level_histograms.txt"))
    for i in (2, 3, 4, 5):
        wl = inputs.make_workload(i, with_feats=False, with_grad=False)
        levels, counts, perm = R.assign_levels(wl.rois, 4, 56.0)
        assert counts.tolist() == [int(v) for v in gold[f"config{i}"]]
        assert counts.tolist() == list(inputs.CONFIGS[i].level_hist)


@pytest.mark.parametrize("K", [0, 1, 5, 1000])
def test_bucketing_is_stable_argsort(K):
    rng = np.random.default_rng(K)
    side = np.exp(rng.uniform(math.log(8), math.log(1200), K))
    rois = np.stack([np.zeros(K), np.zeros(K), np.zeros(K), side, side], 1).astype(np.float32)
    levels, counts, perm = R.assign_levels(rois, 4, 56.0)
    assert counts.sum() == K
    assert np.array_equal(counts, np.bincount(levels, minlength=4))
    assert np.array_equal(perm, np.argsort(levels, kind="stable").astype(np.int32))
    assert sorted(perm.tolist()) == list(range(K))


def test_exact_rational_threshold():
    # With exact rational arithmetic on the fp32 inputs: for a square of fp32 side s the fp32 chain
    # gives sqrt(s*s) == s whenever s*s is exactly representable (small integers), so the level is
    # floor(log2(s/56 + 1e-6)) evaluated on fp32-rounded q.  Check integer sides 1..2000 against a
    # Fraction evaluation of the rounded quantities.
    sides = np.arange(1, 2001, dtype=np.float32)
    rois = np.stack([np.zeros_like(sides)] * 3 + [sides, sides], 1)
    got = R.assign_levels(rois, 4, 56.0)[0]
    for s, lv in zip(sides, got):
        q = np.float32(s) / np.float32(56.0)          # correctly rounded fp32 division
        t = Fraction(float(np.float32(q + np.float32(1e-6))))
        exp = sum(1 for j in (1, 2, 3) if t >= 2 ** j)
        assert lv == exp, (s, lv, exp)
