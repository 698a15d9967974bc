"""Pins of the oracle's kinetic-term path (oracle/aims_oracle.c, block "Kinetic term of h_KS"; Eq. 4, Eq. 24-27
L228-260, Fig. 6a) against facts fixed by mathematics -- never against the CUDA path:
  * closed-form kinetic-energy integrals of s-type Gaussians, <a|-1/2 lap|b> = mu (3 - 2 mu R^2) S_ab, mu = ab/(a+b);
  * lap phi as the trace of the (finite-difference-pinned) Hessian == the radial form (R'' + 2R'/d - l(l+1)R/d^2) Y_lm,
    through batched-and-culled == brute force over all functions and points;
  * the kinetic matrix is symmetric and, up to grid accuracy, equals 1/2 <grad phi_i . grad phi_j> (integration by
    parts; the basis functions vanish smoothly at their cutoff) and is positive semidefinite;
  * kinetic == 0 reduces to O3; the term is additive; invariance under re-batching.
"""
import math

import numpy as np
import pytest

import aims_synth
from aims_synth import bsr_to_dense
from oracle.oracle import Oracle


def test_kinetic_integrals_of_gaussians_match_closed_form():
    alpha = 1.1
    b = aims_synth.make_config(1, n_rad=60, n_ang=302, gaussian_s_only=alpha)
    o = Oracle(b)
    zero = np.zeros(b.n_points)
    T = bsr_to_dense(b, o.integrate_hamiltonian_ks(zero, kinetic=True))
    mu = alpha / 2.0
    for i in range(3):
        for j in range(3):
            R2 = ((b.atom_xyz[i] - b.atom_xyz[j]) ** 2).sum()
            S = (1 / (4 * math.pi)) * (math.pi / (2 * alpha)) ** 1.5 * math.exp(-mu * R2)
            ref = mu * (3.0 - 2.0 * mu * R2) * S
            assert abs(T[i, j] - ref) < 1e-3 * abs(mu * 3.0 * (1 / (4 * math.pi)) * (math.pi / (2 * alpha)) ** 1.5), (i, j, T[i, j], ref)


@pytest.fixture(scope="module")
def toy5():
    b = aims_synth.make_config(5, n_rad=14, n_ang=26, max_batch=40, keep_atoms=6)
    return b, Oracle(b)


def test_batched_hessian_trace_equals_brute_radial_laplacian(toy5, cfg1):
    for b in (cfg1, toy5[0]):
        o = Oracle(b)
        H = bsr_to_dense(b, o.integrate_hamiltonian_ks(b.v, kinetic=True))
        Hb = o.brute_kinetic(b.v)
        assert np.abs(H - Hb).max() <= 1e-12 * np.abs(Hb).max()
        assert np.abs(H - H.T).max() <= 1e-14 * np.abs(H).max()


def test_kinetic_off_reduces_to_plain_hamiltonian_and_term_is_additive(toy5):
    b, o = toy5
    H0 = o.integrate_hamiltonian(b.v, b.g)
    assert np.array_equal(np.isfinite(H0), np.ones_like(H0, dtype=bool))
    Hk0 = o.integrate_hamiltonian_ks(b.v, b.g, kinetic=False)
    assert np.abs(Hk0 - H0).max() <= 1e-13 * np.abs(H0).max()
    Hk = o.integrate_hamiltonian_ks(b.v, b.g, kinetic=True)
    T = o.integrate_hamiltonian_ks(np.zeros(b.n_points), None, kinetic=True)
    assert np.abs(Hk - (H0 + T)).max() <= 1e-12 * np.abs(Hk).max()
    assert np.abs(T).max() > 1e-3


def test_kinetic_matrix_is_half_grad_grad_to_grid_accuracy_and_psd():
    # integration by parts: <i|-1/2 lap|j> = 1/2 <grad i . grad j>; the right-hand side is evaluated from the oracle's own
    # (finite-difference-pinned) gradients on the same grid
    b = aims_synth.make_config(1, n_rad=60, n_ang=302)
    o = Oracle(b)
    T = bsr_to_dense(b, o.integrate_hamiltonian_ks(np.zeros(b.n_points), kinetic=True))
    nb = b.n_basis
    GG = np.zeros((nb, nb))
    for bi in range(b.n_batches):
        idx, phi, dphi = o.eval_basis(bi, want_grad=True)
        w = b.w[b.batch_ptr[bi]:b.batch_ptr[bi + 1]]
        for c in range(3):
            GG[np.ix_(idx, idx)] += 0.5 * (dphi[c] * w) @ dphi[c].T
    scale = np.abs(GG).max()
    assert np.abs(T - GG).max() <= 5e-3 * scale
    assert np.linalg.eigvalsh(0.5 * (T + T.T)).min() >= -5e-3 * scale


def test_kinetic_invariant_under_rebatching():
    a = aims_synth.make_config(1, max_batch=128)
    c = aims_synth.make_config(1, max_batch=37)
    Ha = bsr_to_dense(a, Oracle(a).integrate_hamiltonian_ks(a.v, a.g, kinetic=True))
    Hc = bsr_to_dense(c, Oracle(c).integrate_hamiltonian_ks(c.v, c.g, kinetic=True))
    assert np.abs(Ha - Hc).max() <= 1e-12 * np.abs(Ha).max()


# --------------------------------------------------------------------------- forces with the kinetic operator (Eq. 16)
def test_kinetic_forces_batched_equal_brute_force_and_off_switch(toy5, cfg1):
    for b in (cfg1, toy5[0]):
        o = Oracle(b)
        Dd = bsr_to_dense(b, b.D_values)
        F = o.pulay_forces(b.v, b.D_values, g=b.g, kinetic=True)
        Fb = o.brute_forces(b.v, Dd, g=b.g, kinetic=True)
        assert np.abs(F - Fb).max() <= 1e-12 * np.abs(Fb).max()
        F0 = o.pulay_forces(b.v, b.D_values, g=b.g, kinetic=False)
        Fk = o.pulay_forces(np.zeros(b.n_points), b.D_values, kinetic=True)
        assert np.abs(F - (F0 + Fk)).max() <= 1e-12 * np.abs(F).max()       # the kinetic part is additive
        assert np.abs(Fk).max() > 1e-3


def test_kinetic_forces_are_minus_gradient_of_kinetic_energy_to_grid_accuracy():
    # Eq. 16 relies on the Hermiticity of h_KS; on the grid that holds to quadrature accuracy for -1/2 lap, so the pin is
    # loose in value but catches a wrong sign or factor
    import copy
    b = aims_synth.make_config(1, n_rad=60, n_ang=302)
    o = Oracle(b)
    zero = np.zeros(b.n_points)
    Dd = bsr_to_dense(b, b.D_values)
    F = o.pulay_forces(zero, b.D_values, kinetic=True)

    def energy(xyz):
        b2 = copy.copy(b)
        b2.atom_xyz = np.ascontiguousarray(xyz)
        return float((Dd * bsr_to_dense(b2, Oracle(b2).integrate_hamiltonian_ks(zero, kinetic=True))).sum())

    h = 2e-4
    scale = np.abs(F).max()
    for a, c in ((0, 0), (1, 0), (2, 1)):
        xp, xm = b.atom_xyz.copy(), b.atom_xyz.copy()
        xp[a, c] += h
        xm[a, c] -= h
        fd = -(energy(xp) - energy(xm)) / (2 * h)
        assert abs(fd - F[a, c]) <= 2e-2 * scale, (a, c, fd, F[a, c])


# --------------------------------------------------------------------------- meta-GGA tau matrix (L377, reading P1c)
def test_tau_matrix_with_unit_xi_is_the_kinetic_matrix():
    b = aims_synth.make_config(1, n_rad=60, n_ang=302)
    o = Oracle(b)
    M = bsr_to_dense(b, o.tau_matrix(np.ones(b.n_points)))
    T = bsr_to_dense(b, o.integrate_hamiltonian_ks(np.zeros(b.n_points), kinetic=True))
    scale = np.abs(M).max()
    assert np.abs(M - T).max() <= 5e-3 * scale                  # integration by parts: grid accuracy
    assert np.abs(M - M.T).max() <= 1e-14 * scale
    GG = np.zeros_like(M)
    for bi in range(b.n_batches):
        idx, _, dphi = o.eval_basis(bi, want_grad=True)
        w = b.w[b.batch_ptr[bi]:b.batch_ptr[bi + 1]]
        for c in range(3):
            GG[np.ix_(idx, idx)] += 0.5 * (dphi[c] * w) @ dphi[c].T
    assert np.abs(M - GG).max() <= 1e-12 * scale                # the same sum in another order


def test_tau_matrix_trace_identity_psd_and_additivity(toy5):
    b, o = toy5
    xi = aims_synth.make_xi(b)
    assert xi.min() > 0
    Mv = o.tau_matrix(xi)
    M = bsr_to_dense(b, Mv)
    Dd = bsr_to_dense(b, b.D_values)
    tau = np.zeros(b.n_points)                                  # tau_p = 1/2 sum_ij n_ij grad phi_i . grad phi_j
    for bi in range(b.n_batches):
        idx, _, dphi = o.eval_basis(bi, want_grad=True)
        Db = Dd[np.ix_(idx, idx)]
        tau[b.batch_ptr[bi]:b.batch_ptr[bi + 1]] = 0.5 * sum(((Db @ dphi[c]) * dphi[c]).sum(0) for c in range(3))
    lhs, rhs = float((Dd * M).sum()), float((b.w * xi * tau).sum())
    assert abs(lhs - rhs) <= 1e-11 * max(abs(lhs), abs(rhs), 1.0)
    assert np.linalg.eigvalsh(0.5 * (M + M.T)).min() >= -1e-12 * np.abs(M).max()
    H = o.integrate_hamiltonian(b.v, b.g)
    H2 = o.tau_matrix(xi, H_values=H.copy())
    assert np.abs(H2 - (H + Mv)).max() <= 1e-13 * np.abs(H2).max()     # "added to h^uc_ij"
    half = o.tau_matrix(xi, batches=np.arange(b.n_batches // 2)) + o.tau_matrix(xi, batches=np.arange(b.n_batches // 2, b.n_batches))
    assert np.abs(half - Mv).max() <= 1e-13 * np.abs(Mv).max()
