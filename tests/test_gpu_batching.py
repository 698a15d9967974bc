"""Row f4 (GPU-side batching, reading P12): aims_gpu_batch_points against oracle/batching.py on the same
seeded point clouds.  Exactly one result is correct: batch_ptr and the permutation must be BIT-EXACT.  The clouds are the
configurations' atom-centred grids in a seeded random order (so that nothing of the generator's own batching is left in the
input), plus the degenerate cases: a root that is a batch, n = max + 1, duplicated points, identical points, -0.0, empty."""
import numpy as np
import pytest

import aims_synth
from oracle.batching import batch_points

pytestmark = pytest.mark.gpu


def _gpu(xyz, m):
    import paper_1912_06636_b200 as aims
    order, ptr = aims.aims_gpu_batch_points(xyz, m, device=0)
    return order.cpu().numpy(), ptr


def _shuffled_cloud(cfg, seed=5, **kw):
    bun = aims_synth.make_config(cfg, **kw)
    perm = np.random.default_rng(seed).permutation(bun.n_points)
    return np.ascontiguousarray(bun.xyz[perm]), bun


@pytest.mark.parametrize("cfg,kw,m", [(1, {}, 128), (1, {}, 37), (3, dict(n_rad=8, n_ang=26), 200), (5, dict(n_rad=8, n_ang=26, keep_atoms=30), 64),
                                      (4, dict(n_rad=8, n_ang=38, keep_atoms=40), 500), (2, {}, 200)])
def test_batching_is_bit_exact(cfg, kw, m):
    xyz, bun = _shuffled_cloud(cfg, **kw)
    order, ptr = _gpu(xyz, m)
    o_ref, p_ref = batch_points(xyz, m)
    assert np.array_equal(ptr, p_ref)
    assert np.array_equal(order, o_ref)
    # and the library consumes what it produced: a context over the GPU-batched grid has the oracle's nnz(B) lists
    if bun.n_points < 200000:
        import copy
        import paper_1912_06636_b200 as aims
        from oracle.oracle import Oracle
        b2 = copy.copy(bun)
        b2.xyz = np.ascontiguousarray(xyz[order])
        b2.w = np.ones(len(xyz)); b2.v = np.ones(len(xyz)); b2.g = np.zeros((3, len(xyz)))
        b2.owner = np.zeros(len(xyz), dtype=np.int32)
        b2.batch_ptr = ptr
        ctx = aims.aims_gpu_create(b2, device=0)
        orc = Oracle(b2)
        nnz = ctx.batch_nnz()
        for b in range(0, b2.n_batches, max(1, b2.n_batches // 16)):
            assert nnz[b] == len(orc.batch_nnz(b)[0])
        ctx.close()


def test_batching_degenerate_clouds():
    rng = np.random.default_rng(1)
    for xyz, m in [(rng.standard_normal((5, 3)), 8),                                   # the root is a batch: input order
                   (rng.standard_normal((9, 3)), 8),                                   # n = max + 1
                   (rng.integers(-3, 4, (500, 3)).astype(np.float64) * 0.5, 6),        # lattice: ties and duplicates
                   (np.ones((64, 3)), 6),                                              # identical points: index order
                   (np.zeros((0, 3)), 8)]:
        order, ptr = _gpu(xyz, m)
        o_ref, p_ref = batch_points(xyz, m)
        assert np.array_equal(ptr, p_ref) and np.array_equal(order, o_ref)
    z = np.zeros((40, 3))
    z[::2, 0] = -0.0
    z[:, 1] = np.arange(40) % 3
    order, ptr = _gpu(z, 4)
    o_ref, p_ref = batch_points(z, 4)
    assert np.array_equal(ptr, p_ref) and np.array_equal(order, o_ref)
    import paper_1912_06636_b200 as aims
    with pytest.raises(aims.AimsError):
        _gpu(np.zeros((4, 3)), 0)


def test_batching_config5_full_size():
    """7.9 M points, batches of <= 200 (the benchmark workload): 39,638 batches, bit-exact."""
    xyz, bun = _shuffled_cloud(5)
    order, ptr = _gpu(xyz, 200)
    o_ref, p_ref = batch_points(xyz, 200)
    assert len(ptr) - 1 == bun.n_batches
    assert np.array_equal(ptr, p_ref) and np.array_equal(order, o_ref)
