"""Pins of oracle/batching.py (reading P12 of PAPER.md L210-218) against facts fixed by the definition itself -- never against
the CUDA path, and not against the input generator's own bisection:
  * the result is a permutation cut into batches of <= max points whose sizes follow the stated rule (they depend on n only);
  * replaying the cuts: at every node the children are separated along the axis of largest extent (max of the left <= min of
    the right), and the left child has exactly n_left points;
  * a pure-Python brute force (selection by repeated minimum over (coordinate, index), explicit loops) on tiny clouds,
    including duplicated points and ties in the extents;
  * every batch is sorted by (coordinate, original index) along one axis (the order of the sort that produced it).
"""
import numpy as np
import pytest

from oracle.batching import batch_points, n_left_of


def _sizes(n, m):
    if n <= m:
        return [n]
    nl = n_left_of(n, m)
    return _sizes(nl, m) + _sizes(n - nl, m)


def _brute(xyz, m):
    """Explicit loops only: pick the axis by scanning, pick the n_left smallest by repeated minimum."""
    out, ptr = [], [0]

    def rec(idx):
        if len(idx) <= m:
            out.extend(idx)
            ptr.append(ptr[-1] + len(idx))
            return
        ext = []
        for c in range(3):
            lo = hi = xyz[idx[0]][c]
            for i in idx:
                lo = min(lo, xyz[i][c])
                hi = max(hi, xyz[i][c])
            ext.append(hi - lo)
        ax = 0
        if ext[1] > ext[ax]:
            ax = 1
        if ext[2] > ext[ax]:
            ax = 2
        rest = list(idx)
        srt = []
        while rest:
            best = rest[0]
            for i in rest[1:]:
                if xyz[i][ax] < xyz[best][ax] or (xyz[i][ax] == xyz[best][ax] and i < best):
                    best = i
            rest.remove(best)
            srt.append(best)
        nb = (len(idx) + m - 1) // m
        h = nb // 2
        nl = int(np.floor(h * len(idx) / nb + 0.5))
        rec(srt[:nl])
        rec(srt[nl:])

    rec(list(range(len(xyz))))
    return np.array(out, dtype=np.int64), np.array(ptr, dtype=np.int64)


@pytest.mark.parametrize("n,m", [(1, 4), (4, 4), (5, 4), (37, 5), (200, 7), (513, 64), (1000, 200), (13200, 128)])
def test_cover_sizes_and_rule(n, m):
    rng = np.random.default_rng(n * 31 + m)
    xyz = rng.standard_normal((n, 3)) * np.array([3.0, 1.0, 2.0])
    order, ptr = batch_points(xyz, m)
    assert np.array_equal(np.sort(order), np.arange(n))                  # a permutation: disjoint cover
    sizes = np.diff(ptr)
    assert ptr[0] == 0 and ptr[-1] == n and sizes.max() <= m and sizes.min() >= 1
    assert list(sizes) == _sizes(n, m)
    if n > 10 * m:
        assert sizes.min() >= m - 1 - m // 8                               # "batches of about max points" (P12)


def test_halves_round_up_in_n_left():
    assert n_left_of(5, 4) == 3 and n_left_of(9, 4) == 3 and n_left_of(401, 200) == 134 and n_left_of(400, 200) == 200
    for n in range(5, 400):
        nb = -(-n // 4)
        assert n_left_of(n, 4) == int(np.floor((nb // 2) * n / nb + 0.5))


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_equals_pure_python_brute_force_on_tiny_clouds(seed):
    rng = np.random.default_rng(seed)
    n = [23, 40, 64, 97][seed]
    xyz = rng.integers(-3, 4, (n, 3)).astype(np.float64) * 0.5            # a coarse lattice: many equal coordinates, duplicates
    if seed == 3:
        xyz[:, 1] = xyz[:, 0]                                               # equal extents along x and y: tie -> x
    order, ptr = batch_points(xyz, 6)
    ob, pb = _brute(xyz.tolist(), 6)
    assert np.array_equal(ptr, pb) and np.array_equal(order, ob)


def test_every_cut_separates_along_the_axis_of_largest_extent():
    rng = np.random.default_rng(9)
    xyz = rng.uniform(-1, 1, (3000, 3)) * np.array([1.0, 4.0, 2.0])
    m = 50
    order, ptr = batch_points(xyz, m)

    def check(lo, n):
        if n <= m:
            return
        pts = xyz[order[lo:lo + n]]
        ax = int(np.argmax(pts.max(0) - pts.min(0)))
        nl = n_left_of(n, m)
        assert pts[:nl, ax].max() <= pts[nl:, ax].min()
        check(lo, nl)
        check(lo + nl, n - nl)

    check(0, len(xyz))
    for b in range(len(ptr) - 1):                                           # a batch keeps the order of the sort that made it
        pts = xyz[order[ptr[b]:ptr[b + 1]]]
        idx = order[ptr[b]:ptr[b + 1]]
        ok = False
        for c in range(3):
            k = np.lexsort((idx, pts[:, c]))
            ok |= np.array_equal(k, np.arange(len(idx)))
        assert ok


def test_small_roots_and_degenerate_clouds():
    xyz = np.random.default_rng(4).standard_normal((5, 3))
    order, ptr = batch_points(xyz, 8)
    assert np.array_equal(order, np.arange(5)) and list(ptr) == [0, 5]     # a root that is a batch keeps the input order
    order, ptr = batch_points(np.zeros((0, 3)), 8)
    assert len(order) == 0 and list(ptr) == [0]
    same = np.ones((20, 3))                                                 # all points identical: ties broken by index
    order, ptr = batch_points(same, 6)
    assert np.array_equal(order, np.arange(20))
    z = np.zeros((9, 3))
    z[::2, 0] = -0.0                                                        # -0.0 and +0.0 are the same coordinate
    order, ptr = batch_points(z, 4)
    assert np.array_equal(order, np.arange(9))


def test_generator_batches_follow_the_same_reading():
    """Consistency (not a pin): the bundles the other tests use were batched by the input generator under the same reading."""
    import aims_synth
    bun = aims_synth.make_config(1)
    order, ptr = batch_points(bun.xyz, bun.meta["max_batch"])
    # re-batching an already batched cloud: same tree shape; points keep their batches (the cloud is a permutation of itself)
    assert np.array_equal(ptr, bun.batch_ptr)
    got = [set(map(tuple, bun.xyz[order[ptr[b]:ptr[b + 1]]])) for b in range(len(ptr) - 1)]
    ref = [set(map(tuple, bun.xyz[bun.batch_ptr[b]:bun.batch_ptr[b + 1]])) for b in range(bun.n_batches)]
    assert got == ref
