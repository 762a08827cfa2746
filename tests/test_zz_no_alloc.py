"""noit_quadtree_balance_static (`-m gpu`): the balance pass whose scratch is a file-scope device
array of libnoit.so instead of context memory -- for callers that cannot cudaMalloc (CUDA-graph
capture, tight serving loops).  Collected LAST on purpose (the suite runs with pytest -x).

Checked against the existing path (noit_quadtree_balance) on two calls in a row -- the second call
finds the first call's contents in the shared array -- and against the oracle; every output of the
pass is an integer class (bit-exact) except the fp32 scales (1e-6, as in test_steps_gpu.py).  The
test also shows that the call allocates nothing through torch's allocator and that the size limit is
an error code, and it passes alone in a fresh process as well as after the other tests.
"""
import numpy as np
import pytest
import torch

import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def noit():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_16747_b200 as m
    return m


def u32(t):
    return t.cpu().numpy().view(np.uint32)


def random_valid_masks(rng, n):
    """21-bit masks with child bit => parent bit (include/noit.h mask layout)."""
    out = np.zeros(n, np.uint32)
    for i in range(n):
        m = 0
        if rng.random() < 0.5:
            m |= 1
            for c in range(4):
                if rng.random() < 0.5:
                    m |= 1 << (1 + c)
                    for g in range(4):
                        if rng.random() < 0.4:
                            m |= 1 << (5 + 4 * c + g)
        out[i] = m
    return out


def empty_out(W, H, dev="cuda"):
    Tx, Ty = (W + 63) // 64, (H + 63) // 64
    cx, cy = (W + 7) // 8, (H + 7) // 8
    return dict(tile_level=torch.empty(Tx * Ty, dtype=torch.uint8, device=dev),
                cell_level=torch.empty(cx * cy, dtype=torch.uint8, device=dev),
                hist=torch.empty(4, dtype=torch.int32, device=dev),
                scales=torch.empty(3, dtype=torch.float32, device=dev))


def same(a, b, ref):
    for k in ("tile_mask", "hist"):
        assert np.array_equal(u32(a[k]), u32(b[k])), k
        assert np.array_equal(u32(a[k]), ref[k]), k
    for k in ("tile_level", "cell_level"):
        assert torch.equal(a[k], b[k]), k
        assert np.array_equal(a[k].cpu().numpy(), ref[k]), k
    assert torch.equal(a["scales"], b["scales"])                      # same kernel, same inputs: same bits
    assert np.max(np.abs(a["scales"].cpu().numpy().astype(np.float64) - ref["scales"])) <= 1e-6


def test_balance_static_equals_the_allocating_path_twice_in_a_row(noit):
    ctx = noit.Noit()
    # two calls in a row, different frames and sizes: the second finds the first one's masks,
    # ticket and accumulators in the shared array (a larger frame first, then a smaller one)
    for seed, W, H, k in ((0, 3840, 2160, 2), (1, 1920, 1080, 2), (2, 1000, 700, 5), (3, 40, 40, 2)):
        rng = np.random.default_rng(seed)
        Tx, Ty = (W + 63) // 64, (H + 63) // 64
        m = random_valid_masks(rng, Tx * Ty)
        ref = oracle.quadtree_balance(m, W, H, iterations=k)
        d_a = torch.from_numpy(m.view(np.int32).copy()).cuda()
        d_b = d_a.clone()
        out_b = empty_out(W, H)
        a = ctx.quadtree_balance(d_a, W, H, iterations=k)                               # existing path
        torch.cuda.synchronize()
        before = torch.cuda.memory_stats()["allocation.all.allocated"]
        b = ctx.quadtree_balance(d_b, W, H, iterations=k, out=out_b, static_scratch=True)
        after = torch.cuda.memory_stats()["allocation.all.allocated"]
        assert after == before, "the static-scratch call allocated device memory through torch"
        same(a, b, ref)
        # the same frame again, straight after: stale contents of the array must not matter
        d_c = torch.from_numpy(m.view(np.int32).copy()).cuda()
        c = ctx.quadtree_balance(d_c, W, H, iterations=k, out=empty_out(W, H), static_scratch=True)
        same(a, c, ref)
    # a second context shares the array (stream-ordered calls: no race)
    ctx2 = noit.Noit()
    rng = np.random.default_rng(9)
    m = random_valid_masks(rng, 30 * 17)
    ref = oracle.quadtree_balance(m, 1920, 1080)
    a = ctx.quadtree_balance(torch.from_numpy(m.view(np.int32).copy()).cuda(), 1920, 1080)
    b = ctx2.quadtree_balance(torch.from_numpy(m.view(np.int32).copy()).cuda(), 1920, 1080,
                              out=empty_out(1920, 1080), static_scratch=True)
    same(a, b, ref)


def test_balance_static_rejects_sizes_beyond_its_scratch(noit):
    ctx = noit.Noit()
    W, H = 64 * 129, 64 * 128                                       # 16512 base tiles > 16384
    mask = torch.zeros(129 * 128, dtype=torch.int32, device="cuda")
    keep = mask.clone()
    with pytest.raises(noit.NoitError) as e:
        ctx.quadtree_balance(mask, W, H, out=empty_out(W, H), static_scratch=True)
    assert e.value.status == 2 and "16384" in str(e.value)           # NOIT_ERR_SIZE, limit named
    assert torch.equal(mask, keep)                                   # nothing was launched
    W, H = 64 * 128, 64 * 128                                        # exactly at the limit: accepted
    m = random_valid_masks(np.random.default_rng(4), 128 * 128)
    ref = oracle.quadtree_balance(m, W, H)
    b = ctx.quadtree_balance(torch.from_numpy(m.view(np.int32).copy()).cuda(), W, H, out=empty_out(W, H),
                             static_scratch=True)
    assert np.array_equal(u32(b["tile_mask"]), ref["tile_mask"]) and np.array_equal(u32(b["hist"]), ref["hist"])
