"""Worker of tests/test_steps_gpu.py::test_bounds_checked_build_counts_no_violation: runs with
NOIT_LIBRARY = libnoit_debug.so (the staged resolve kernel compiled with -DNOIT_DEBUG_BOUNDS; our
own memcheck, compute-sanitizer being closed on the GPU pool).  Every staging regime of the kernel
is exercised and compared with the oracle; the violation counter must stay 0 -- and must move when
a deliberately malformed CSR makes the last tile reach past the arrays."""
import json
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))
import noit_scenes  # noqa: E402
import oracle  # noqa: E402
import paper_2606_16747_b200 as noit  # noqa: E402
from noit_scenes.raster import FragBuf  # noqa: E402
from test_parity_gpu import BG, check_resolve, random_fb  # noqa: E402


def main():
    assert noit.lib_path() and os.environ.get("NOIT_LIBRARY", "").endswith("libnoit_debug.so")
    cases = 0
    w = noit_scenes.mlp_weights(7)
    ctx = noit.Noit(w, 1)
    ctx32 = noit.Noit(w, 0)
    # dense tiles at every staging boundary (light / depth-only chunks / colour chunks / cold path)
    for dtype, lo, hi in ((np.float16, 100, 128), (np.float32, 100, 128), (np.float16, 180, 188),
                          (np.float32, 150, 157), (np.float16, 60, 70), (np.float32, 36, 40), (np.float16, 28, 32)):
        rng = np.random.default_rng(lo * 1000 + hi)
        W, H = 96, 5
        counts = rng.integers(lo, hi + 1, W * H)
        off = np.zeros(W * H + 1, np.uint32)
        off[1:] = np.cumsum(counts)
        F = int(off[-1])
        fbh = FragBuf(W, H, off, rng.uniform(0.01, 0.99, F).astype(np.float32), rng.uniform(0, 1, (F, 4)).astype(dtype))
        check_resolve(noit, fbh, w, 1, ctx.resolve(noit.DeviceFragBuf.from_host(fbh), BG))
        cases += 1
    # ragged random frames: odd sizes, empty pixels, lists far above the cap, both precisions
    rng = np.random.default_rng(5)
    for _ in range(16):
        W, H = int(rng.integers(1, 90)), int(rng.integers(1, 30))
        max_n = int(rng.choice([1, 3, 12, 40, 130, 300]))
        dtype = np.float16 if rng.random() < 0.6 else np.float32
        heavy = (int(rng.integers(1, 6)), int(rng.choice([200, 700, 1700]))) if rng.random() < 0.5 else None
        fbh = random_fb(rng, W, H, max_n, dtype, tie_frac=0.3, empty_frac=float(rng.choice([0.0, 0.2, 0.7])), heavy=heavy)
        p = int(rng.integers(0, 2))
        check_resolve(noit, fbh, w, p, (ctx if p else ctx32).resolve(noit.DeviceFragBuf.from_host(fbh), BG))
        cases += 1
    # a whole config: cfg2 (all light tiles) and a 448x264 cfg4 through the adaptive and pixel-list modes
    sc = noit_scenes.cfg2(0)
    c2 = noit.Noit(sc.weights, sc.mlp_precision)
    check_resolve(noit, sc.full, sc.weights, sc.mlp_precision, c2.resolve(noit.DeviceFragBuf.from_host(sc.full), BG))
    s4 = noit_scenes.cfg4(0, W=448, H=264, n_prims=96, mean_band=(10.0, 12.0), cap=64)
    f4, h4, q4 = (noit.DeviceFragBuf.from_host(b) for b in (s4.full, s4.half, s4.quarter))
    c4 = noit.Noit(s4.weights, s4.mlp_precision)
    p4 = c4.resolve(f4, BG)
    qt = c4.quadtree(p4["final"], 448, 264, 0, 6)
    c4.resolve(f4, BG, half=h4, quarter=q4, cell_level=qt["cell_level"])
    plist = torch.arange(0, 448 * 264, 7, dtype=torch.int32, device="cuda")
    c4.resolve(f4, BG, out=p4, pixel_list=plist, pixel_count=torch.tensor([plist.numel()], dtype=torch.int32, device="cuda"))
    from test_oracle_pins import _weights931
    c4.resolve_dfaoit(f4, _weights931(1), BG)
    cases += 5
    clean = sum(c.debug_bounds_violations() for c in (ctx, ctx32, c2, c4))
    # the counter is live: a CSR whose last offset overshoots F by 3 makes the frame's last tile reach
    # past the arrays (3 fragments, inside the allocator's padding)
    sc1 = noit_scenes.cfg1(0)
    off = sc1.full.offsets.copy()
    off[-1] += 3
    d = noit.DeviceFragBuf.from_host(sc1.full)
    bad = noit.DeviceFragBuf(d.width, d.height, torch.from_numpy(off.view(np.int32)).cuda(), d.depth, d.rgba)
    cb = noit.Noit(sc1.weights, sc1.mlp_precision)
    cb.resolve(bad, BG)
    fired = cb.debug_bounds_violations()
    print(json.dumps({"cases": cases, "violations": clean, "fired_on_malformed_csr": fired}))


if __name__ == "__main__":
    main()
