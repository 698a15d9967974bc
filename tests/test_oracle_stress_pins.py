"""Pins of the oracle's Pulay-stress path (oracle/aims_oracle.c, block O9; Eq. 20) against facts
fixed by mathematics -- never against the CUDA path:
  * V sigma_lm = d/d eps_lm [ Tr(D H(eps)) - Tr(Q S(eps)) ] by central differences of the already pinned H and S
    (tests/test_oracle_pins.py) on a homogeneously strained copy of the inputs: atoms and grid points r -> (1 + eps) r,
    with D, Q, v, g and the weights fixed (reading P22);
  * batched-and-culled == the term-by-term brute force (every strained factor differentiated separately);
  * for a uniform translation of the whole system nothing changes; for an s-only basis without the GGA term sigma is
    symmetric (the integrand is d_l d_m R'(d)/d); the trace of V sigma equals the derivative under isotropic scaling;
  * linear in (D, Q), 1/V scaling, invariant under re-batching;
  * kinetic != 0 (the Pulay part of the kinetic stress): batched-and-culled with the Hessian-trace Laplacian == brute force with the
    radial-form Laplacian and both index orders; additive in (v, kinetic); and, through the commutator [t, x_m d_l] = -d_l d_m,
    sigma(0, kin) + sum_ij n_ij <phi_i| d_l d_m |phi_j> == central differences of Tr(n t(eps)) of the pinned kinetic matrix, to
    grid accuracy (the bar tests/test_oracle_kinetic_pins.py uses for the kinetic forces).
"""
import copy

import numpy as np
import pytest

import aims_synth
from aims_synth import bsr_to_dense, make_q_values
from oracle.oracle import Oracle


@pytest.fixture(scope="module")
def toy5():
    b = aims_synth.make_config(5, n_rad=14, n_ang=26, max_batch=40, keep_atoms=6)
    return b, Oracle(b)


def _strained(b, eps):
    """Copy of the bundle with atoms and points mapped by r -> (1 + eps) r; everything attached to points is kept."""
    b2 = copy.copy(b)
    A = np.eye(3) + eps
    b2.atom_xyz = np.ascontiguousarray(b.atom_xyz @ A.T)
    b2.xyz = np.ascontiguousarray(b.xyz @ A.T)
    return b2


def _energy(b, D_dense, Q_dense, use_g, eps):
    b2 = _strained(b, eps)
    o2 = Oracle(b2)
    H = bsr_to_dense(b2, o2.integrate_hamiltonian(b.v, b.g if use_g else None))
    e = float((D_dense * H).sum())
    if Q_dense is not None:
        S = bsr_to_dense(b2, o2.integrate_hamiltonian(np.ones(b.n_points)))
        e -= float((Q_dense * S).sum())
    return e


@pytest.mark.parametrize("case", ["cfg1_lda", "cfg1_gga_q", "toy5_gga_q", "toy5_lda_q"])
def test_pulay_stress_is_strain_derivative_of_the_energy(case, toy5, cfg1):
    b = cfg1 if case.startswith("cfg1") else toy5[0]
    use_g = "gga" in case
    use_q = case.endswith("_q")
    o = Oracle(b)
    Qv = make_q_values(b) if use_q else None
    Dd = bsr_to_dense(b, b.D_values)
    Qd = bsr_to_dense(b, Qv) if use_q else None
    sig = o.pulay_stress(b.v, b.D_values, g=b.g if use_g else None, Q_values=Qv, volume=1.0)
    scale = np.abs(sig).max()
    assert scale > 1e-3
    h = 1e-4
    comps = [(0, 0), (1, 2), (2, 1), (2, 2), (0, 1)] if b.n_atoms > 3 else [(l, m) for l in range(3) for m in range(3)]
    for (l, m) in comps:
        e = np.zeros((3, 3))
        e[l, m] = h
        fd = (_energy(b, Dd, Qd, use_g, e) - _energy(b, Dd, Qd, use_g, -e)) / (2 * h)
        assert abs(fd - sig[l, m]) <= 5e-6 * scale, (l, m, fd, sig[l, m])


@pytest.mark.parametrize("use_g", [False, True])
def test_batched_stress_equals_brute_force(toy5, cfg1, use_g):
    for b in (cfg1, toy5[0]):
        o = Oracle(b)
        Qv = make_q_values(b)
        g = b.g if use_g else None
        sig = o.pulay_stress(b.v, b.D_values, g=g, Q_values=Qv, volume=3.5)
        sb = o.brute_stress(b.v, bsr_to_dense(b, b.D_values), g=g, Q_dense=bsr_to_dense(b, Qv), volume=3.5)
        assert np.abs(sig - sb).max() <= 1e-12 * np.abs(sb).max()
        s2 = o.pulay_stress(b.v, 2.0 * b.D_values, g=g, Q_values=2.0 * Qv, volume=7.0)      # linear in (D, Q), 1/V
        assert np.abs(s2 - sig).max() <= 1e-13 * np.abs(sig).max()
        # without q
        s0 = o.pulay_stress(b.v, b.D_values, g=g, volume=3.5)
        sb0 = o.brute_stress(b.v, bsr_to_dense(b, b.D_values), g=g, volume=3.5)
        assert np.abs(s0 - sb0).max() <= 1e-12 * np.abs(sb0).max()


def test_trace_is_the_derivative_under_isotropic_scaling_and_translation_changes_nothing(toy5):
    b, o = toy5
    Qv = make_q_values(b)
    Dd, Qd = bsr_to_dense(b, b.D_values), bsr_to_dense(b, Qv)
    sig = o.pulay_stress(b.v, b.D_values, g=b.g, Q_values=Qv)
    h = 1e-4
    fd = (_energy(b, Dd, Qd, True, h * np.eye(3)) - _energy(b, Dd, Qd, True, -h * np.eye(3))) / (2 * h)
    assert abs(fd - np.trace(sig)) <= 5e-6 * np.abs(sig).max()
    # rigid translation of atoms and points: distance vectors, hence sigma, unchanged (to rounding of the coordinates)
    t = np.array([3.25, -1.5, 7.125])
    b2 = copy.copy(b)
    b2.atom_xyz = np.ascontiguousarray(b.atom_xyz + t)
    b2.xyz = np.ascontiguousarray(b.xyz + t)
    s2 = Oracle(b2).pulay_stress(b.v, b.D_values, g=b.g, Q_values=Qv)
    assert np.abs(s2 - sig).max() <= 1e-9 * np.abs(sig).max()


def test_s_only_lda_stress_is_symmetric():
    b = aims_synth.make_config(1, gaussian_s_only=0.9)
    o = Oracle(b)
    rng = np.random.default_rng(5)
    C = rng.standard_normal((b.n_basis, 2))
    from aims_synth import dense_to_bsr
    Dv = dense_to_bsr(b, C @ C.T)
    sig = o.pulay_stress(b.v, Dv)
    assert np.abs(sig).max() > 1e-4
    assert np.abs(sig - sig.T).max() <= 1e-12 * np.abs(sig).max()
    # and it equals -1/2 sum_at (R_at - c) x F_at-like sum rule only for pair terms; here just check against brute force
    sb = o.brute_stress(b.v, C @ C.T)
    assert np.abs(sig - sb).max() <= 1e-12 * np.abs(sb).max()


def test_stress_invariant_under_rebatching():
    a = aims_synth.make_config(1, max_batch=128)
    c = aims_synth.make_config(1, max_batch=37)
    sa = Oracle(a).pulay_stress(a.v, a.D_values, g=a.g, Q_values=make_q_values(a))
    sc = Oracle(c).pulay_stress(c.v, c.D_values, g=c.g, Q_values=make_q_values(c))
    assert np.abs(sa - sc).max() <= 1e-12 * np.abs(sa).max()


# --------------------------------------------------------------------------- kinetic branch (h_KS phi_j carries -1/2 lap phi_j)
@pytest.mark.parametrize("use_g", [False, True])
def test_kinetic_stress_batched_equals_brute_force_and_is_additive(toy5, cfg1, use_g):
    for b in (cfg1, toy5[0]):
        o = Oracle(b)
        Qv = make_q_values(b)
        g = b.g if use_g else None
        Dd, Qd = bsr_to_dense(b, b.D_values), bsr_to_dense(b, Qv)
        sig = o.pulay_stress(b.v, b.D_values, g=g, Q_values=Qv, kinetic=True, volume=3.5)
        sb = o.brute_stress(b.v, Dd, g=g, Q_dense=Qd, kinetic=True, volume=3.5)      # radial-form Laplacian, no batches, no culling
        assert np.abs(sig - sb).max() <= 1e-12 * np.abs(sb).max()
        s_off = o.pulay_stress(b.v, b.D_values, g=g, Q_values=Qv, kinetic=False, volume=3.5)
        s_kin = o.pulay_stress(np.zeros(b.n_points), b.D_values, kinetic=True, volume=3.5)
        assert np.abs(s_kin).max() > 1e-3 * np.abs(sig).max()                         # the branch contributes
        assert np.abs(sig - (s_off + s_kin)).max() <= 1e-12 * np.abs(sig).max()       # and is additive
        sk_b = o.brute_stress(np.zeros(b.n_points), Dd, kinetic=True, volume=3.5)
        assert np.abs(s_kin - sk_b).max() <= 1e-12 * np.abs(sk_b).max()


def test_kinetic_stress_plus_commutator_term_is_the_strain_derivative_of_the_kinetic_energy():
    """E(eps) = Tr(n t(eps)) on the strained grid = sum_p w_p sum_ij n_ij phi_i (t phi_j).  Its derivative has the Pulay part the
    oracle returns, 2 sum w n_ij (d_l phi_i)(r - R_i)_m (t phi_j), and the derivative of the factor t phi_j, which by Hermiticity of
    t and [t, x_m d_l] = -d_l d_m equals the Pulay part again plus C_lm = sum_ij n_ij <phi_i| d_l d_m |phi_j>.  C is evaluated here
    from the oracle's finite-difference-pinned Hessian of the density: phi_i d_l d_m phi_j summed with n_ij is
    hess_n[lm] / 2 - sum_ij n_ij d_l phi_i d_m phi_j.  Hermiticity holds on the grid to quadrature accuracy only, hence the loose
    bar -- but a wrong sign or factor in the kinetic branch is an error of the order of the scale itself."""
    b = aims_synth.make_config(1, n_rad=60, n_ang=302)
    o = Oracle(b)
    zero = np.zeros(b.n_points)
    Dd = bsr_to_dense(b, b.D_values)
    P = o.pulay_stress(zero, b.D_values, kinetic=True)
    hess = o.density_hessian(b.D_values)                                   # [6][n]: xx, yy, zz, xy, xz, yz
    hx = [[0, 3, 4], [3, 1, 5], [4, 5, 2]]
    C = np.zeros((3, 3))
    for bi in range(b.n_batches):
        idx, phi, dphi = o.eval_basis(bi, want_grad=True)
        sl = slice(b.batch_ptr[bi], b.batch_ptr[bi + 1])
        Db = Dd[np.ix_(idx, idx)]
        for l in range(3):
            for m in range(3):
                gg = np.einsum("ip,ij,jp->p", dphi[l], Db, dphi[m])
                C[l, m] += (b.w[sl] * (0.5 * hess[hx[l][m]][sl] - gg)).sum()

    def energy(eps):
        b2 = _strained(b, eps)
        return float((Dd * bsr_to_dense(b2, Oracle(b2).integrate_hamiltonian_ks(zero, kinetic=True))).sum())

    h = 2e-4
    scale = np.abs(P).max()
    assert np.abs(C).max() > 0.3 * scale                                   # the commutator term is not a detail
    for (l, m) in [(0, 0), (1, 1), (0, 1), (1, 0), (2, 1)]:
        e = np.zeros((3, 3))
        e[l, m] = h
        fd = (energy(e) - energy(-e)) / (2 * h)
        assert abs(fd - (P[l, m] + C[l, m])) <= 2e-2 * scale, (l, m, fd, P[l, m], C[l, m])
        assert abs(fd - (-P[l, m] + C[l, m])) > 2e-2 * scale or abs(P[l, m]) < 2e-2 * scale     # a sign slip would be seen
