"""Cross-check of the two CPU statements of the path against each other: the plain triple-loop oracle
(oracle/aims_oracle.c) and the paper-style per-batch BLAS form of Fig. 6's CPU column (oracle/blas_baseline.py: one matmul pair
per batch).  Different arithmetic order and a library dgemm on one side, the written-out loops on
the other: they must agree to <= 1e-12.  Neither touches the CUDA path."""
import numpy as np
import pytest

import aims_synth
from aims_synth import dense_to_bsr
from oracle.blas_baseline import BlasBaseline
from oracle.oracle import Oracle


@pytest.mark.parametrize("case", ["cfg1", "cfg3_coarse", "cfg5_toy"])
def test_blas_form_equals_plain_oracle(case):
    bun = {"cfg1": lambda: aims_synth.make_config(1),
           "cfg3_coarse": lambda: aims_synth.make_config(3, n_rad=6, n_ang=14, keep_atoms=24),
           "cfg5_toy": lambda: aims_synth.make_config(5, n_rad=8, n_ang=14, keep_atoms=12)}[case]()
    orc, bl = Oracle(bun), BlasBaseline(bun)
    for g in (None, bun.g):
        H = dense_to_bsr(bun, bl.hamiltonian_dense(bun.v, g))
        ref = orc.integrate_hamiltonian(bun.v, g)
        assert np.linalg.norm(H - ref) <= 1e-12 * np.linalg.norm(ref)
    n, gn = bl.density(bl.dense(bun.D_values), want_grad=True)
    n_ref, gn_ref = orc.update_density(bun.D_values, want_grad=True)
    assert np.abs(n - n_ref).max() <= 1e-12 * np.abs(n_ref).max()
    assert np.abs(gn - gn_ref).max() <= 1e-12 * np.abs(gn_ref).max()
    # a sub-list of batches, as bench.py samples them
    sel = np.arange(0, bun.n_batches, 3)
    Hs = dense_to_bsr(bun, bl.hamiltonian_dense(bun.v, bun.g, batches=sel))
    refs = orc.integrate_hamiltonian(bun.v, bun.g, batches=sel)
    assert np.linalg.norm(Hs - refs) <= 1e-12 * np.linalg.norm(refs)
