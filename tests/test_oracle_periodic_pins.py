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


# ---- geometry of reading P23 (oracle/periodic.py): image enumeration and the point map
def _cell_samples(lat, m=7):
    g = (np.arange(m) + 0.5) / m
    f = np.array([[a, b, c] for a in g for b in g for c in g])
    corners = np.array([[a, b, c] for a in (0.0, 1.0) for b in (0.0, 1.0) for c in (0.0, 1.0)])
    return np.concatenate([f, corners]) @ lat


@pytest.mark.parametrize("case", ["toy", "si"])
def test_image_list_is_a_superset_of_every_atom_within_reach_and_is_ordered(case):
    from oracle.periodic import periodic_images
    b = aims_synth.make_periodic(n_rad=6, n_ang=10) if case == "toy" else aims_synth.make_periodic_si(n_cells=2, n_rad=4, n_ang=6)
    reach = b.rcut
    home, n = periodic_images(b.lattice, b.frac, reach)
    keys = set((int(h), int(a), int(bb), int(c)) for h, (a, bb, c) in zip(home, n))
    assert len(keys) == len(home)                                            # no atom twice
    assert np.all(n[: b.n_home] == 0) and np.array_equal(home[: b.n_home], np.arange(b.n_home))   # the cell's own atoms first
    rest = [(int(a), int(bb), int(c), int(h)) for h, (a, bb, c) in zip(home[b.n_home:], n[b.n_home:])]
    assert rest == sorted(rest)
    # brute force over a large integer box: every periodic atom closer than `reach` to a sample point of the cell is listed
    samples = _cell_samples(b.lattice)
    R = 4
    for a in range(b.n_home):
        for n1 in range(-R, R + 1):
            for n2 in range(-R, R + 1):
                for n3 in range(-R, R + 1):
                    pos = (b.frac[a] + np.array([n1, n2, n3])) @ b.lattice
                    if np.linalg.norm(samples - pos, axis=1).min() < reach:
                        assert (a, n1, n2, n3) in keys
    # ... and the list is not wildly larger than needed: every listed atom is within reach + cell diagonal of the cell centre
    centre = np.array([0.5, 0.5, 0.5]) @ b.lattice
    diag = np.linalg.norm(b.lattice.sum(axis=0)) + np.linalg.norm(b.lattice[0] - b.lattice[1]) + np.linalg.norm(b.lattice[2])
    pos = (b.frac[home] + n) @ b.lattice
    assert np.linalg.norm(pos - centre, axis=1).max() < 2.0 * reach + diag
    # the seeded periodic bundle (whose Bloch sums are pinned by the Gaussian lattice sums above) uses exactly this list
    assert np.array_equal(home, b.atom_home) and np.allclose(n @ b.lattice, b.atom_T, rtol=0, atol=1e-12)


def test_wrapped_points_differ_by_a_lattice_vector_and_lie_in_the_cell():
    from oracle.periodic import inverse_lattice, wrap_points
    b = aims_synth.make_periodic(n_rad=10, n_ang=14)
    lat = b.lattice
    assert np.abs(inverse_lattice(lat) @ lat - np.eye(3)).max() < 1e-14
    assert np.abs(inverse_lattice(lat) - np.linalg.inv(lat)).max() < 1e-15
    r = b.xyz_unwrapped
    w = wrap_points(lat, r)
    shift = (r - w) @ np.linalg.inv(lat)
    assert np.abs(shift - np.rint(shift)).max() < 1e-11                      # an integer combination of a_1, a_2, a_3
    assert np.abs(np.rint(shift)).max() >= 1                                 # some points really were outside
    f = w @ np.linalg.inv(lat)
    assert f.min() > -1e-12 and f.max() < 1.0 + 1e-12
    assert np.abs(wrap_points(lat, w) - w).max() < 1e-12                     # idempotent
    assert np.abs(w - b.xyz).max() < 1e-12                                   # the bundle's (pinned) points
    # a point on a lattice translate of r0 maps onto the image of r0
    r0 = np.array([[0.3, 0.2, 0.1]]) @ lat
    for nvec in ([1, 0, 0], [-2, 3, 1], [0, -1, 4]):
        assert np.abs(wrap_points(lat, r0 + np.array(nvec) @ lat) - r0).max() < 1e-12


def test_wrap_of_a_point_a_hair_below_a_cell_face_stays_inside_the_half_open_cell():
    """Reading P23 promises fractional coordinates in [0, 1).  For f = -1e-20 the difference f - floor(f) = 1 - 1e-20 rounds to
    1.0, the excluded face; that face is the f = 0 face of the neighbouring cell, so the wrapped point must sit at f = 0
    exactly (cubic cell of edge 4: coordinates 0, not 4).  Points well inside and exactly on faces keep their textbook images."""
    from oracle.periodic import wrap_points
    lat = 4.0 * np.eye(3)
    tiny = 1e-20
    r = np.array([[-tiny, 1.0, 2.0], [1.0, -tiny, -tiny], [4.0, 8.0, -4.0], [-1.0, 5.0, 3.5], [-4.0 * 2.0 ** -60, 0.5, 0.5]])
    w = wrap_points(lat, r)
    want = np.array([[0.0, 1.0, 2.0], [1.0, 0.0, 0.0], [0.0, 0.0, 0.0], [3.0, 1.0, 3.5], [0.0, 0.5, 0.5]])
    assert np.array_equal(w, want)
    f = w / 4.0
    assert f.min() >= 0.0 and f.max() < 1.0
    assert np.array_equal(wrap_points(lat, w), w)          # idempotent to the bit
