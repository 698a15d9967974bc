"""Plain statement of the cut-plane batching of PAPER.md L210-218 under DESIGN.md reading P12 -- the oracle of
aims_gpu_batch_points.  TEST INFRASTRUCTURE, NOT THE PRODUCT; imports nothing from paper_1912_06636_b200 and nothing from the
input generator's C helper (aims_synth/_heavy.c has its own copy of the recipe: an input generator, not a reference).

The paper: the grid is cut "into spatially compact sets of points" by a "grid adapted cut-plane method" ("Algorithm 3 of [37]"),
"until some targeted number of points per subset is reached" (L210-212); it does not state the algorithm.  Reading P12:
  a set of n points is a batch if n <= max_pts; otherwise, with nb = ceil(n / max_pts), the n_left = round(floor(nb/2) n / nb)
  (halves up) points smallest in (coordinate along the axis of largest extent -- ties to x, then y --, original index) are the
  left child, the rest the right child; children are processed depth-first, left first; a batch keeps the order of the
  sort that produced it (the root, if it is itself a batch, keeps the input order).
Pins (tests/test_oracle_batching_pins.py): permutation / cover / size rule, every cut separates its children along the axis
of largest extent, a pure-Python selection-by-repeated-minimum brute force on tiny clouds, ties and duplicates.
"""
import numpy as np


def n_left_of(n, max_pts):
    nb = -(-n // max_pts)
    h = nb // 2
    return (2 * h * n + nb) // (2 * nb)          # round(h n / nb), halves up, in integers


def batch_points(xyz, max_pts):
    """(order, batch_ptr): order[k] = original index of the point at position k; batch_ptr [n_batches + 1]."""
    xyz = np.asarray(xyz, dtype=np.float64).reshape(-1, 3)
    n = len(xyz)
    order, ptr = [], [0]

    def rec(idx):
        m = len(idx)
        if m <= max_pts:
            order.append(idx)
            ptr.append(ptr[-1] + m)
            return
        pts = xyz[idx]
        ext = pts.max(axis=0) - pts.min(axis=0)
        ax = int(np.argmax(ext))                  # first maximum: ties to x, then y
        srt = np.lexsort((idx, pts[:, ax]))       # primary key: coordinate; secondary: original index
        idx = idx[srt]
        nl = n_left_of(m, max_pts)
        rec(idx[:nl])
        rec(idx[nl:])

    if n:
        rec(np.arange(n, dtype=np.int64))
    return (np.concatenate(order) if order else np.zeros(0, dtype=np.int64)), np.array(ptr, dtype=np.int64)
