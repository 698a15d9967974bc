"""Pins of the periodic path (oracle/aims_oracle.c, block "Periodic boundary conditions"; Eq. 6-8, 11-12, L113-115)
against facts fixed by mathematics -- never against the CUDA path:
  * the grid of the cell atoms, mapped back into the cell with periodic partition weights, integrates 1 to the cell volume;
  * s_ij(k) of s-type Gaussians = sum_T e^{ik.T} S_free(R_i - R_j - T), the closed-form lattice sum;
  * the fold equals a direct quadrature of Eq. 8 with explicitly built Bloch functions chi_ik (Eq. 7);
  * h(k), s(k) Hermitian, real at k = 0, s(k) positive definite.
"""
import math

import numpy as np
import pytest

import aims_synth
from oracle.oracle import Oracle

KPTS = [np.zeros(3), np.array([0.31, -0.17, 0.23]), np.array([0.7, 0.2, -0.4])]


def test_mapped_grid_integrates_to_cell_volume():
    b = aims_synth.make_periodic(n_rad=60, n_ang=302)
    fr = b.xyz @ np.linalg.inv(b.lattice)
    assert fr.min() >= 0.0 and fr.max() < 1.0
    assert abs(b.w.sum() / abs(np.linalg.det(b.lattice)) - 1.0) < 3e-4
    assert b.w.min() >= 0.0


def test_overlap_of_gaussians_matches_closed_form_lattice_sum():
    alpha = 1.1
    b = aims_synth.make_periodic(n_rad=60, n_ang=302, gaussian_s_only=alpha)
    o = Oracle(b)
    S_uc = o.integrate_hamiltonian(np.ones(b.n_points))
    pref = (1 / (4 * math.pi)) * (math.pi / (2 * alpha)) ** 1.5
    R = b.atom_xyz[:b.n_home]
    rng = range(-4, 5)
    for k in KPTS:
        S = o.bloch_fold(S_uc, b.atom_home, b.atom_T, b.n_home, k)
        for i in range(b.n_home):
            for j in range(b.n_home):
                ref = 0.0
                for n1 in rng:
                    for n2 in rng:
                        for n3 in rng:
                            T = np.array([n1, n2, n3]) @ b.lattice
                            d2 = ((R[i] - R[j] - T) ** 2).sum()
                            ref += np.exp(1j * (k @ T)) * pref * math.exp(-alpha * d2 / 2)
                assert abs(S[i, j] - ref) < 1e-3 * pref, (k, i, j, S[i, j], ref)


@pytest.fixture(scope="module")
def per():
    b = aims_synth.make_periodic(n_rad=16, n_ang=26, max_batch=60)
    return b, Oracle(b)


def test_fold_equals_direct_quadrature_with_bloch_functions(per):
    b, o = per
    H_uc = o.integrate_hamiltonian(b.v)
    nfn = int(b.atom_fn_ptr[1])
    nhb = b.n_home * nfn
    # phi of every periodic atom at every point, through the oracle's (pinned) evaluation
    phi = np.zeros((b.n_atoms * nfn, b.n_points))
    for bi in range(b.n_batches):
        idx, ph, _ = o.eval_basis(bi)
        phi[idx, b.batch_ptr[bi]:b.batch_ptr[bi + 1]] = ph
    for k in KPTS:
        chi = np.zeros((nhb, b.n_points), dtype=complex)
        for A in range(b.n_atoms):
            chi[b.atom_home[A] * nfn:(b.atom_home[A] + 1) * nfn] += np.exp(1j * (k @ b.atom_T[A])) * phi[A * nfn:(A + 1) * nfn]
        ref = (chi.conj() * (b.w * b.v)) @ chi.T
        H = o.bloch_fold(H_uc, b.atom_home, b.atom_T, b.n_home, k)
        assert np.abs(H - ref).max() <= 1e-12 * np.abs(ref).max()


def test_folded_matrices_are_hermitian_and_overlap_is_positive_definite(per):
    b, o = per
    S_uc = o.integrate_hamiltonian(np.ones(b.n_points))
    H_uc = o.integrate_hamiltonian(b.v, b.g)
    for k in KPTS:
        S = o.bloch_fold(S_uc, b.atom_home, b.atom_T, b.n_home, k)
        H = o.bloch_fold(H_uc, b.atom_home, b.atom_T, b.n_home, k)
        assert np.abs(S - S.conj().T).max() <= 1e-14 * np.abs(S).max()
        assert np.abs(H - H.conj().T).max() <= 1e-14 * np.abs(H).max()
        assert np.linalg.eigvalsh(S).min() > 0.0
        if not k.any():
            assert np.abs(S.imag).max() == 0.0 and np.abs(H.imag).max() == 0.0
        else:
            assert np.abs(S.imag).max() > 1e-6
