"""Host-side logic: roofline byte accounting against the oracle's sample enumeration, and the
multi-rank (shard-by-image) path on CPU with the gloo backend, world_size 2."""
import os
import socket

import numpy as np
import pytest

from oracle import raf_ref as R
import bench_roofline as roofline
from paper_1906_07155_b200 import inputs, sharding


@pytest.mark.parametrize("index", [2, 4])
def test_roofline_footprint_matches_oracle_enumeration(index):
    wl = inputs.make_workload(index, with_feats=False, with_grad=False)
    cfg = wl.cfg
    fp = roofline.footprint(wl.rois, cfg.level_shapes, cfg.scales, cfg.out_size, 2, True, 56.0)
    shapes = [(s[0], 1, s[2], s[3]) for s in cfg.level_shapes]
    masks = R.footprint(shapes, cfg.scales, wl.rois, cfg.out_size, 2, True)
    assert fp["union_px"] == sum(int(m.sum()) for m in masks)
    assert fp["level_hist"] == list(cfg.level_hist)
    assert fp["union_px"] <= fp["per_roi_px"] <= fp["requested_px"]


def test_algorithmic_bytes_config2_matches_survey_table():
    wl = inputs.make_workload(2, with_feats=False, with_grad=False)
    cfg = wl.cfg
    fp = roofline.footprint(wl.rois, cfg.level_shapes, cfg.scales, cfg.out_size, 2, True, 56.0)
    ab = roofline.algorithmic_bytes(fp, cfg.K, 256, (7, 7), 4, 4, 4)
    # B_f = 118.7 + 51.4 = 170.1 MB, B_b = 51.4 + 182.8 = 234.2 MB
    assert abs(ab["fwd"] / 1e6 - 170.1) < 0.1
    assert abs(ab["bwd"] / 1e6 - 234.2) < 0.1


def test_image_ranges_partition():
    for n_img in (1, 2, 5, 16):
        for world in (1, 2, 3, 8):
            spans = [sharding.image_range(n_img, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n_img
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = inputs.make_workload(5, n_img=4, per_img=12, channels=4)
        cfg = wl.cfg
        rois = wl.rois.copy()
        rois[5, 0] = 9           # invalid image: owned by nobody
        local, rows = sharding.shard_rois(rois, cfg.n_img, rank, world)
        lo, hi = sharding.image_range(cfg.n_img, rank, world)
        feats = [f[lo:hi] for f in wl.feats]
        out_local = R.forward(feats, cfg.scales, local, (7, 7), 2, True, 56.0)
        # the ONLY communication of the job: barrier + max-over-ranks of the local time
        dist.barrier()
        ms = sharding.max_over_ranks_ms(10.0 + rank, dist)
        q.put((rank, rows, out_local, ms))
    finally:
        dist.destroy_process_group()


def test_shard_by_image_world2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=180) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = inputs.make_workload(5, n_img=4, per_img=12, channels=4)
    rois = wl.rois.copy()
    rois[5, 0] = 9
    full = R.forward(wl.feats, wl.cfg.scales, rois, (7, 7), 2, True, 56.0)
    merged = np.zeros_like(full)
    seen = []
    for rank, rows, out_local, ms in res:
        merged[rows] = out_local
        seen += rows.tolist()
        assert ms == 11.0                      # max over ranks
    assert sorted(seen) == [k for k in range(48) if k != 5]
    assert np.array_equal(merged, full)        # no exchange needed: shards are independent
