"""CPU-side checks of the boundary (`-m "not gpu"`): libnoit.so loads and exports every symbol
include/noit.h declares, the ctypes structs match the header layout, the host-side sharding logic
is right, and a world_size-2 gloo run of the N>1 plumbing works.  No compute calls here."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "noit.h")


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(noit_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_exported():
    import paper_2606_16747_b200 as noit
    L = noit.lib()
    syms = declared_symbols()
    assert set(syms) == set(noit.EXPORTS), (syms, noit.EXPORTS)
    for s in syms:
        assert getattr(L, s) is not None
    # the dynamic symbol table agrees (nm is part of binutils)
    out = subprocess.run(["nm", "-D", "--defined-only", noit.lib_path()], capture_output=True, text=True)
    if out.returncode == 0:
        exported = {l.split()[-1] for l in out.stdout.splitlines() if l.strip()}
        assert set(syms) <= exported


def test_struct_layout_matches_header(tmp_path):
    """sizeof/offsetof from a tiny C program compiled against noit.h == the ctypes structs."""
    from paper_2606_16747_b200 import binding as B
    prog = tmp_path / "layout.c"
    prog.write_text(r'''
#include <stdio.h>
#include <stddef.h>
#include "noit.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu\n", sizeof(noit_fragbuf), sizeof(noit_layers), sizeof(noit_resolve_desc),
         sizeof(noit_qt_params), sizeof(noit_reproject_desc));
  printf("%zu %zu %zu %zu\n", offsetof(noit_resolve_desc, cell_level), offsetof(noit_resolve_desc, background),
         offsetof(noit_resolve_desc, pixel_list), offsetof(noit_resolve_desc, out_depth1));
  printf("%zu %zu %zu\n", offsetof(noit_reproject_desc, depth_threshold),
         offsetof(noit_reproject_desc, prev_trans), offsetof(noit_reproject_desc, reject_count));
  return 0; }''')
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(prog), "-o", str(exe)])
    lines = subprocess.check_output([str(exe)], text=True).split("\n")
    sizes = [int(v) for v in lines[0].split()]
    assert sizes == [C.sizeof(B.FragBufC), C.sizeof(B.LayersC), C.sizeof(B.ResolveDescC),
                     C.sizeof(B.QtParamsC), C.sizeof(B.ReprojectDescC)]
    R = B.ResolveDescC
    assert [int(v) for v in lines[1].split()] == [R.cell_level.offset, R.background.offset,
                                                  R.pixel_list.offset, R.out_depth1.offset]
    J = B.ReprojectDescC
    assert [int(v) for v in lines[2].split()] == [J.depth_threshold.offset, J.prev_trans.offset,
                                                  J.reject_count.offset]


def test_product_does_not_import_oracle():
    """The product path never routes through the oracle (no import, no dlopen of it)."""
    pkg = os.path.join(ROOT, "paper_2606_16747_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "noit_oracle" not in txt, f


def test_shard_rows_balanced_and_covering():
    from paper_2606_16747_b200.sharding import gather_rows, shard_rows, slice_rows
    rng = np.random.default_rng(0)
    W, H = 96, 300
    counts = rng.integers(0, 9, W * H)
    counts[: W * 100] *= 4                       # heavy top: bands must not be equal-height
    off = np.zeros(W * H + 1, np.uint32)
    off[1:] = np.cumsum(counts)
    depth = rng.random(int(off[-1])).astype(np.float32)
    rgba = rng.random((int(off[-1]), 4)).astype(np.float16)
    for ws in (1, 2, 3, 8):
        bands = shard_rows(off, W, H, ws)
        assert len(bands) == ws and bands[0][0] == 0 and bands[-1][1] == H
        for (a0, a1), (b0, b1) in zip(bands[:-1], bands[1:]):
            assert a1 == b0 and a0 <= a1
        for y0, y1 in bands[:-1]:
            assert y1 % 64 == 0
        parts = []
        for y0, y1 in bands:
            o, d, c = slice_rows(off, depth, rgba, W, y0, y1)
            assert o[0] == 0 and o[-1] == d.shape[0] == c.shape[0]
            assert np.array_equal(np.diff(o.astype(np.int64)), counts[y0 * W:y1 * W])
            parts.append(np.diff(o.astype(np.int64)).astype(np.float32))
        assert np.array_equal(gather_rows(parts, bands, W, H, 1), counts.astype(np.float32))
    b2 = shard_rows(off, W, H, 2)
    assert b2[0][1] < H // 2                      # fragment-balanced: the heavy band is shorter


def test_bench_gloo_world2(tmp_path):
    """N>1 plumbing (rank env, barrier, max-over-ranks reduce, rank-0-only JSON) on CPU/gloo."""
    env = dict(os.environ, NOIT_BENCH_DRYRUN="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29731", os.path.join(ROOT, "bench.py"),
           "--gpus", "2", "--steps", "2", "--warmup", "1"]
    out = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout
    rec = json.loads(lines[0])
    assert rec["n_gpus"] == 2 and rec["dryrun"] is True and rec["scaling"] == "weak"
    assert rec["ranks_seen"] == 2


def test_sharded_path_gloo_world2():
    """SURVEY 8(e) with two real ranks (gloo, CPU): each rank slices ITS band of the same seeded
    frame (shard_rows / slice_rows), exchanges the reprojection halo with its neighbour
    (exchange_halo_rows) and rank 0 reassembles per-band results with gather_rows."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29741",
           os.path.join(ROOT, "tests", "gloo_shard_worker.py")]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-3000:]
    import json
    rec = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert rec["world"] == 2 and rec["counts_equal"] and rec["first_depth_equal"] and rec["halo_ok"]
    (a0, a1), (b0, b1) = rec["bands"]
    assert a0 == 0 and a1 == b0 and b1 == 256 and a1 % 64 == 0 and 0 < a1 < 256
    f = rec["fragments_per_rank"]
    assert abs(f[0] - f[1]) <= 0.5 * sum(f)                   # balanced by fragments, 64-row granularity


def test_band_matrix_is_the_frame_matrix_in_band_coordinates():
    """band_matrix: a point of the band, mapped by the band's matrix in the band's NDC, lands where
    the frame's matrix puts it in the frame's NDC (float64 check of the coordinate bookkeeping)."""
    from paper_2606_16747_b200.sharding import band_matrix
    import noit_scenes
    H, y0, y1 = 1080, 256, 640
    proj = noit_scenes.perspective(60.0, 16 / 9, 0.1, 100.0)
    M = (proj @ noit_scenes.view_matrix(np.zeros(3), 0.0, 0.0)) @ np.linalg.inv(
        proj @ noit_scenes.view_matrix(np.array([0.1, -0.05, 0.2]), 0.01, -0.02))
    Mb = band_matrix(M, H, y0, y1)
    rng = np.random.default_rng(0)
    for _ in range(50):
        yl, xn, d = rng.uniform(0, y1 - y0), rng.uniform(-1, 1), rng.uniform(0.9, 0.999)
        c = Mb @ np.array([xn, 2 * (yl + 0.5) / (y1 - y0) - 1, d, 1.0])
        g = M @ np.array([xn, 2 * (yl + y0 + 0.5) / H - 1, d, 1.0])
        # previous row inside the band's own frame vs inside the whole frame
        rb = (c[1] / c[3] + 1) * 0.5 * (y1 - y0) + y0
        rg = (g[1] / g[3] + 1) * 0.5 * H
        assert abs(rb - rg) < 1e-9 and abs(c[0] / c[3] - g[0] / g[3]) < 1e-12 and abs(c[2] / c[3] - g[2] / g[3]) < 1e-12


def test_bench_reference_arm_contract():
    """`bench.py --impl reference` (the oracle on the host cores): one JSON line with the contract's
    keys, BASELINE.json's metric string, and a cpu_baseline that describes the run."""
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout
    rec = json.loads(lines[0])
    want = json.load(open(os.path.join(ROOT, "BASELINE.json")))["metric"]
    assert rec["impl"] == "reference" and rec["metric"] == want and rec["unit"] == "Mpixels/s"
    assert rec["value"] > 0 and rec["higher_is_better"] is True and rec["vs_baseline"] is None
    assert rec["steps"] == 1 and rec["n_gpus"] == 1 and rec["data"] == "synthetic"
    assert rec["cpu_baseline"]["kind"] == "oracle" and rec["cpu_baseline"]["cores"] >= 1
    assert rec["cpu_baseline"]["value"] == rec["value"] and rec["cpu_baseline"]["sample"]
    assert rec["e2e"] == {"value": rec["value"], "unit": "Mpixels/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert rec["config"]["workload"].startswith("cfg3") and rec["gpu_launches"] == 0
