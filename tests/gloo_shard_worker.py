"""Worker of tests/test_abi.py::test_sharded_path_gloo_world2 (launched by torch.distributed.run,
backend gloo, CPU): every rank REALLY takes its band of the same seeded frame through
shard_rows / slice_rows, computes a per-pixel stand-in on it (the fragment counts -- no arithmetic of
the method runs on the CPU), exchanges its reprojection halo with its neighbours, and rank 0
reassembles the frame with gather_rows and checks the rank -> band mapping."""
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import noit_scenes  # noqa: E402
from paper_2606_16747_b200.sharding import (exchange_halo_rows, extended_band, gather_rows, halo_rows,  # noqa: E402
                                            shard_rows, slice_rows)


def main():
    dist.init_process_group(backend="gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    sc = noit_scenes.cfg2(0, W=320, H=256, n_prims=32)
    fb = sc.full
    W, H = fb.width, fb.height
    bands = shard_rows(fb.offsets, W, H, world)
    y0, y1 = bands[rank]
    off, depth, rgba = slice_rows(fb.offsets, fb.depth, fb.rgba, W, y0, y1)
    assert off[0] == 0 and off[-1] == depth.shape[0] == rgba.shape[0]
    counts = np.diff(off.astype(np.int64)).astype(np.float32)
    first_depth = np.where(counts > 0, depth[np.minimum(off[:-1], max(depth.shape[0] - 1, 0))], 1.0).astype(np.float32)
    gathered = [None] * world
    dist.all_gather_object(gathered, (rank, (y0, y1), counts, first_depth))
    # halo exchange on a "previous frame" whose pixel (y, x) carries y * W + x
    prev = torch.arange(H * W, dtype=torch.float32).reshape(H, W, 1)
    halo = halo_rows(H)                                       # ceil(0.02 * 256) + 1 = 7
    above, below = exchange_halo_rows(prev[y0:y1].clone(), halo, rank, world)
    e0, e1 = extended_band((y0, y1), halo, H)
    ok_halo = True
    if rank > 0:
        ok_halo &= above is not None and torch.equal(above, prev[y0 - above.shape[0]:y0]) and y0 - above.shape[0] == e0
    else:
        ok_halo &= above is None and e0 == 0
    if rank < world - 1:
        ok_halo &= below is not None and torch.equal(below, prev[y1:y1 + below.shape[0]]) and y1 + below.shape[0] == e1
    else:
        ok_halo &= below is None and e1 == H
    flags = [None] * world
    dist.all_gather_object(flags, bool(ok_halo))
    if rank == 0:
        gathered.sort(key=lambda g: g[0])
        assert [g[1] for g in gathered] == bands
        full_counts = gather_rows([g[2] for g in gathered], bands, W, H, 1)
        full_d1 = gather_rows([g[3] for g in gathered], bands, W, H, 1)
        want = np.diff(fb.offsets.astype(np.int64)).astype(np.float32)
        start = np.minimum(fb.offsets[:-1], fb.depth.shape[0] - 1)
        want_d1 = np.where(want > 0, fb.depth[start], 1.0).astype(np.float32)
        print(json.dumps({"world": world, "bands": bands, "counts_equal": bool(np.array_equal(full_counts, want)),
                          "first_depth_equal": bool(np.array_equal(full_d1, want_d1)), "halo_ok": all(flags),
                          "halo": halo, "fragments_per_rank": [int(g[2].sum()) for g in gathered]}))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
