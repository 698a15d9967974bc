"""Host-side sharding of the batch loops over GPUs (every batch belongs to one task and "at no time does any
process know the full grid"; L231: the batch sums are trivially parallel; Eq. 28-29: one sum of H over tasks is the
only communication step; L312: the density needs none).  Bookkeeping only -- no arithmetic of the method lives here.

A rank's context is created over ITS OWN batches only (points, per-batch lists and workspaces scale with 1/N):
  1. first_phase_range: an equal-count contiguous range per rank; the rank creates a throw-away context over that slice and
     reads |nnz(B)| of its batches (aims_gpu_batch_nnz);
  2. the per-batch costs n_p * nnz^2 are summed over ranks (one tiny all-reduce), partition_batches cuts the depth-first batch
     order into contiguous ranges of equal cost (spatially compact per GPU, so each GPU touches a bounded part of H);
  3. slice_bundle(bun, b0, b1) is the rank's input, aims_gpu_create runs on it, H_values (global pattern) is all-reduced once.
"""
import copy

import numpy as np


def partition_batches(cost, n_parts):
    """Contiguous ranges [lo, hi) of (almost) equal total cost; cost[b] >= 0."""
    nb = len(cost)
    csum = np.concatenate([[0.0], np.cumsum(np.asarray(cost, dtype=np.float64))])
    bounds = [0]
    for r in range(1, n_parts):
        target = csum[-1] * r / n_parts
        bounds.append(int(np.clip(np.searchsorted(csum, target, side="left"), bounds[-1], nb)))
    bounds.append(nb)
    return [(bounds[r], bounds[r + 1]) for r in range(n_parts)]


def first_phase_range(n_batches, rank, world):
    """Equal-count contiguous range of batches for the cost probe."""
    return (n_batches * rank) // world, (n_batches * (rank + 1)) // world


# attributes that describe the whole system (atoms, basis, block pattern, matrices): every rank keeps them whole, also when one
# of their dimensions happens to equal the number of grid points
GLOBAL_FIELDS = frozenset((
    "atom_xyz", "atom_species", "species_shell_ptr", "shell_l", "shell_rcut", "shell_spline", "spline_coef", "shell_zeta",
    "shell_norm", "row_ptr", "col_atom", "blk_off", "blk_ld", "D_values", "atom_fn_ptr", "batch_ptr",
    "lattice", "frac", "atom_home", "atom_n", "atom_T"))


def slice_bundle(bun, b0, b1):
    """The inputs of batches [b0, b1) only.  batch_ptr is cut and rebased to 0; EVERY other array attribute that carries one
    entry per grid point -- leading dimension n_points ([n], [n][k]: xyz, w, v, owner, xyz_unwrapped, ...) or, for two-dimensional
    component-major fields, trailing dimension n_points ([k][n]: g) -- is cut to the batches' point range, whatever its name, so
    that a per-point field added to the bundle later cannot stay full-size beside a shrunken grid.  GLOBAL_FIELDS (atoms, basis,
    block pattern, D: objects every rank needs whole) and non-array attributes are shared unchanged.
    Returns (sliced bundle, first point, last point)."""
    n = int(bun.xyz.shape[0])
    lo, hi = int(bun.batch_ptr[b0]), int(bun.batch_ptr[b1])
    s = copy.copy(bun)
    s.batch_ptr = np.ascontiguousarray(bun.batch_ptr[b0:b1 + 1] - lo).astype(np.int64)
    for name, val in vars(bun).items():
        if name in GLOBAL_FIELDS or not isinstance(val, np.ndarray) or val.ndim == 0:
            continue
        if val.shape[0] == n:
            setattr(s, name, np.ascontiguousarray(val[lo:hi]))
        elif val.ndim == 2 and val.shape[1] == n:
            setattr(s, name, np.ascontiguousarray(val[:, lo:hi]))
    return s, lo, hi
