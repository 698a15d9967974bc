"""Pins of the CPU oracle (oracle/aims_oracle.c) against facts fixed by mathematics, library routines and brute
force -- never against itself and never against the CUDA path.  The paper (arXiv:1912.06636) prints no numerical
value for this path, so every pin is mathematical; see DESIGN.md "Oracle pins".
All tests here run on the CPU (-m "not gpu").
"""
import math

import numpy as np
import pytest

import aims_synth
from aims_synth import bsr_to_dense
from oracle import oracle as orc
from oracle.oracle import Oracle


# --------------------------------------------------------------------------- Y_lm (reading P10)
def _real_ylm_scipy(l, m, theta, phi):
    """Orthonormal real harmonics without Condon-Shortley phase from scipy's complex Y_l^m (library routine)."""
    from scipy.special import sph_harm_y
    if m == 0:
        return sph_harm_y(l, 0, theta, phi).real
    y = sph_harm_y(l, abs(m), theta, phi)
    s = math.sqrt(2.0) * (-1.0) ** abs(m)
    return s * (y.real if m > 0 else y.imag)


def test_ylm_matches_scipy_library():
    rng = np.random.default_rng(1)
    for _ in range(50):
        u = rng.standard_normal(3)
        u /= np.linalg.norm(u)
        theta, phi = math.acos(u[2]), math.atan2(u[1], u[0])
        for l in range(4):
            Y = orc.solid_harmonics(l, u)
            ref = np.array([_real_ylm_scipy(l, m, theta, phi) for m in range(-l, l + 1)])
            assert np.abs(Y - ref).max() < 5e-15


def test_ylm_orthonormal_exact_quadrature():
    # Gauss-Legendre in cos(theta) x uniform phi integrates products of l<=3 harmonics exactly
    x, wx = np.polynomial.legendre.leggauss(8)
    nphi = 16
    ph = 2 * np.pi * np.arange(nphi) / nphi
    rows = []
    wts = []
    for xi, wi in zip(x, wx):
        for p in ph:
            s = math.sqrt(1 - xi * xi)
            u = np.array([s * math.cos(p), s * math.sin(p), xi])
            rows.append(np.concatenate([orc.solid_harmonics(l, u) for l in range(4)]))
            wts.append(wi * 2 * np.pi / nphi)
    Y = np.array(rows)
    G = Y.T @ (Y * np.array(wts)[:, None])
    assert np.abs(G - np.eye(16)).max() < 1e-14


def test_solid_harmonic_gradient_finite_difference_and_homogeneity():
    rng = np.random.default_rng(2)
    h = 1e-6
    for _ in range(20):
        r = rng.standard_normal(3)
        for l in range(4):
            Y, G = orc.solid_harmonics(l, r, want_grad=True)
            # homogeneous of degree l: S(2r) = 2^l S(r); Euler: r.grad S = l S
            assert np.allclose(orc.solid_harmonics(l, 2 * r), 2.0 ** l * Y, rtol=1e-14, atol=1e-14)
            assert np.allclose(G @ r, l * Y, rtol=1e-13, atol=1e-13)
            for c in range(3):
                e = np.zeros(3)
                e[c] = h
                fd = (orc.solid_harmonics(l, r + e) - orc.solid_harmonics(l, r - e)) / (2 * h)
                assert np.abs(fd - G[:, c]).max() < 1e-8 * max(1.0, np.abs(G).max())


# --------------------------------------------------------------------------- radial spline (reading P8)
def test_radial_spline_matches_scipy_cubicspline(cfg1, cfg1_oracle):
    from scipy.interpolate import CubicSpline
    b, o = cfg1, cfg1_oracle
    rk = b.r0 * np.exp(b.log_inc * np.arange(b.n_knots))
    rng = np.random.default_rng(3)
    for s in range(len(b.shell_l)):
        table = aims_synth.radial_analytic(rk, b.shell_l[s], b.shell_zeta[s], b.shell_rcut[s], b.shell_norm[s])
        cs = CubicSpline(np.arange(b.n_knots, dtype=float), table, bc_type="natural")
        # knots reproduce the table
        for k in (0, 1, 57, 150, b.n_knots - 2):
            R, _ = o.radial(s, rk[k] * (1 + 1e-15))
            assert abs(R - table[k]) <= 1e-12 * max(1.0, abs(table[k]))
        for d in np.exp(rng.uniform(np.log(b.r0), np.log(rk[-1]), 200)):
            t = math.log(d / b.r0) / b.log_inc
            R, dR = o.radial(s, d)
            assert abs(R - cs(t)) <= 1e-12 * max(1.0, abs(cs(t)))
            ref_d = cs(t, 1) / (b.log_inc * d)            # chain rule dt/dd = 1/(log_inc d)
            assert abs(dR - ref_d) <= 1e-10 * max(1.0, abs(ref_d))
        # the spline follows the analytic function it was tabulated from (O(h^4))
        for d in (0.3, 1.0, 2.5, 4.2):
            R, _ = o.radial(s, d)
            ana = aims_synth.radial_analytic(np.array([d]), b.shell_l[s], b.shell_zeta[s], b.shell_rcut[s], b.shell_norm[s])[0]
            assert abs(R - ana) < 2e-4 * max(abs(ana), 1e-3)
    # below the first knot the function is held at r0 (reading P11)
    assert o.radial(0, 0.0)[0] == o.radial(0, b.r0)[0]


# --------------------------------------------------------------------------- O1: phi and grad phi
@pytest.fixture(scope="module")
def toy5():
    """first 6 atoms of config 5 (Bi/Se shells up to l = 3) on a coarse grid"""
    b = aims_synth.make_config(5, n_rad=14, n_ang=26, max_batch=40, keep_atoms=6)
    return b, Oracle(b)


def test_phi_is_radial_times_ylm_and_zero_beyond_cutoff(toy5):
    b, o = toy5
    rng = np.random.default_rng(4)
    sh = 0
    for a in range(b.n_atoms):
        sp = b.atom_species[a]
        for s in range(b.species_shell_ptr[sp], b.species_shell_ptr[sp + 1]):
            l = b.shell_l[s]
            u = rng.standard_normal(3)
            u /= np.linalg.norm(u)
            d = rng.uniform(0.05, b.shell_rcut[s] * 0.999)
            phi = o.shell_at_point(a, s, b.atom_xyz[a] + d * u, want_grad=False)
            R, _ = o.radial(s, d)
            assert np.allclose(phi, R * orc.solid_harmonics(l, u), rtol=1e-11, atol=1e-14)
            out, gout = o.shell_at_point(a, s, b.atom_xyz[a] + (b.shell_rcut[s] + 1e-9) * u)
            assert np.all(out == 0.0) and np.all(gout == 0.0)
            sh += 1
    assert sh > 10


def test_grad_phi_matches_central_finite_difference(toy5):
    b, o = toy5
    rng = np.random.default_rng(5)
    h = 1e-5
    worst = 0.0
    for a in range(b.n_atoms):
        sp = b.atom_species[a]
        for s in range(b.species_shell_ptr[sp], b.species_shell_ptr[sp + 1]):
            for d in (0.02, 0.7, 3.1, b.shell_rcut[s] - 0.3):      # near nucleus, mid, inside the cutoff ramp
                u = rng.standard_normal(3)
                u /= np.linalg.norm(u)
                r = b.atom_xyz[a] + d * u
                phi, gr = o.shell_at_point(a, s, r)
                scale = max(np.abs(gr).max(), np.abs(phi).max(), 1e-6)
                for c in range(3):
                    e = np.zeros(3)
                    e[c] = h
                    fd = (o.shell_at_point(a, s, r + e, False) - o.shell_at_point(a, s, r - e, False)) / (2 * h)
                    worst = max(worst, np.abs(fd - gr[:, c]).max() / scale)
    assert worst < 2e-7


# --------------------------------------------------------------------------- grid, weights, batches (inputs)
def test_partition_weights_sum_to_one_at_every_point(cfg1):
    b = cfg1
    rng = np.random.default_rng(6)
    pts = np.concatenate([b.xyz[rng.integers(0, b.n_points, 400)], rng.uniform(-3, 3, (400, 3))])
    tot = np.zeros(len(pts))
    for a in range(b.n_atoms):
        wa = aims_synth.partition_weights(b.atom_xyz, pts, np.full(len(pts), a, dtype=np.int32), b.meta["r_part"])
        assert wa.min() >= 0.0 and wa.max() <= 1.0
        tot += wa
    assert np.abs(tot - 1.0).max() < 1e-14


def test_partition_weights_sum_to_one_dense_cluster():
    b = aims_synth.make_config(2, n_rad=6, n_ang=14)
    rng = np.random.default_rng(7)
    pts = b.xyz[rng.integers(0, b.n_points, 300)]
    tot = sum(aims_synth.partition_weights(b.atom_xyz, pts, np.full(len(pts), a, dtype=np.int32), b.meta["r_part"])
              for a in range(b.n_atoms))
    assert np.abs(tot - 1.0).max() < 1e-13


def test_single_centre_gaussian_integral_closed_form():
    b = aims_synth.make_config(1, keep_atoms=1)
    r2 = ((b.xyz - b.atom_xyz[0]) ** 2).sum(1)
    for alpha in (0.5, 1.0, 3.0, 8.0):
        num = (b.w * np.exp(-alpha * r2)).sum()
        assert abs(num / (math.pi / alpha) ** 1.5 - 1.0) < 1e-6    # 40 log-radial shells (trapezoid in s)


def test_batches_are_a_disjoint_cover_within_size(cfg1):
    b = cfg1
    n = np.diff(b.batch_ptr)
    assert b.batch_ptr[0] == 0 and b.batch_ptr[-1] == b.n_points and n.min() >= 1 and n.max() <= 128
    # the permutation applied by the generator is a bijection onto the unbatched grid
    ref = aims_synth.make_config(1, max_batch=10 ** 9)
    key = lambda x: np.lexsort((x[:, 2], x[:, 1], x[:, 0]))  # noqa: E731
    assert np.array_equal(b.xyz[key(b.xyz)], ref.xyz[key(ref.xyz)])
    assert abs(b.w.sum() - ref.w.sum()) < 1e-9 * ref.w.sum()
    # compactness: a batch is far smaller than the cloud
    ext = max(np.ptp(b.xyz[b.batch_ptr[i]:b.batch_ptr[i + 1]], axis=0).max() for i in range(b.n_batches))
    assert ext < np.ptp(b.xyz, axis=0).max()


# --------------------------------------------------------------------------- O2: nnz(B)
def test_nnz_lists_against_brute_distance_matrix(toy5):
    b, o = toy5
    fn_atom = np.repeat(np.arange(b.n_atoms), np.diff(b.atom_fn_ptr))
    fn_rc = np.concatenate([np.repeat(b.shell_rcut[s], 2 * b.shell_l[s] + 1)
                            for a in range(b.n_atoms)
                            for s in range(b.species_shell_ptr[b.atom_species[a]], b.species_shell_ptr[b.atom_species[a] + 1])])
    assert np.array_equal(o.atom_fn_ptr, b.atom_fn_ptr)
    sizes = set()
    for bi in range(b.n_batches):
        pts = b.xyz[b.batch_ptr[bi]:b.batch_ptr[bi + 1]]
        dmin = np.linalg.norm(pts[:, None, :] - b.atom_xyz[None, :, :], axis=2).min(0)
        idx = o.batch_nnz(bi)[0]
        assert np.all(np.diff(idx) > 0)
        listed = np.zeros(b.n_basis, dtype=bool)
        listed[idx] = True
        margin = 1e-9
        assert np.all(listed[dmin[fn_atom] < fn_rc - margin])        # everything that touches is listed
        assert not np.any(listed[dmin[fn_atom] > fn_rc + margin])    # nothing out of reach is listed
        sizes.add(len(idx))
    assert len(sizes) > 1                                            # culling really varies over batches


# --------------------------------------------------------------------------- O3: H and S
def test_overlap_of_gaussians_matches_closed_form():
    alpha = 1.1
    b = aims_synth.make_config(1, n_rad=60, n_ang=302, gaussian_s_only=alpha)
    o = Oracle(b)
    S = bsr_to_dense(b, o.integrate_hamiltonian(np.ones(b.n_points)))
    for i in range(3):
        for j in range(3):
            R2 = ((b.atom_xyz[i] - b.atom_xyz[j]) ** 2).sum()
            ref = (1 / (4 * math.pi)) * (math.pi / (2 * alpha)) ** 1.5 * math.exp(-alpha * R2 / 2)
            assert abs(S[i, j] / ref - 1.0) < 3e-4


def test_hamiltonian_of_gaussians_matches_three_centre_closed_form():
    # v is a sum of atom-centred Gaussians (aims_synth recipe), so <i|v|j> is a sum of three-centre Gaussian integrals
    alpha = 0.9
    b = aims_synth.make_config(1, n_rad=60, n_ang=302, gaussian_s_only=alpha)
    o = Oracle(b)
    H = bsr_to_dense(b, o.integrate_hamiltonian(b.v))
    c, al = b.meta["v_c"], b.meta["v_alpha"]
    for i in range(3):
        for j in range(i, 3):
            A, B = b.atom_xyz[i], b.atom_xyz[j]
            ref = 0.0
            for a in range(3):
                for k in range(3):
                    gsum = 2 * alpha + al[a, k]
                    P = (alpha * A + alpha * B + al[a, k] * b.atom_xyz[a]) / gsum
                    expo = (alpha * (A @ A) + alpha * (B @ B) + al[a, k] * (b.atom_xyz[a] @ b.atom_xyz[a])) - gsum * (P @ P)
                    ref += c[a, k] * (math.pi / gsum) ** 1.5 * math.exp(-expo)
            ref /= 4 * math.pi
            assert abs(H[i, j] / ref - 1.0) < 5e-4
            assert H[i, j] == pytest.approx(H[j, i], rel=1e-13)


def test_overlap_symmetric_positive_definite_and_normalised(cfg1, cfg1_oracle):
    b, o = cfg1, cfg1_oracle
    S = bsr_to_dense(b, o.integrate_hamiltonian(np.ones(b.n_points)))
    assert np.abs(S - S.T).max() < 1e-14
    np.linalg.cholesky(S)
    assert np.abs(np.diag(S) - 1.0).max() < 2e-3           # radial functions are L2-normalised by the generator


def test_overlap_positive_definite_dense_cluster():
    b = aims_synth.make_config(2, n_rad=16, n_ang=50, keep_atoms=10)
    o = Oracle(b)
    S = bsr_to_dense(b, o.integrate_hamiltonian(np.ones(b.n_points)))
    assert np.abs(S - S.T).max() < 1e-13
    assert np.linalg.eigvalsh(S).min() > 0


@pytest.mark.parametrize("use_g", [False, True])
def test_batched_culled_equals_brute_force(toy5, cfg1, cfg1_oracle, use_g):
    for b, o in (toy5, (cfg1, cfg1_oracle)):
        g = b.g if use_g else None
        H = bsr_to_dense(b, o.integrate_hamiltonian(b.v, g))
        Dd = bsr_to_dense(b, b.D_values)
        n, gn = o.update_density(b.D_values, want_grad=True)
        Hb, nb, gnb = o.brute(b.v, g, Dd, want_grad=True)
        assert np.linalg.norm(H - Hb) <= 1e-13 * np.linalg.norm(Hb)
        assert np.abs(n - nb).max() <= 1e-13 * np.abs(nb).max()
        assert np.abs(gn - gnb).max() <= 1e-13 * np.abs(gnb).max()
        assert np.abs(Hb - Hb.T).max() <= 1e-13 * np.abs(Hb).max()


def test_result_is_invariant_under_rebatching():
    a = aims_synth.make_config(1, max_batch=128)
    c = aims_synth.make_config(1, max_batch=37)
    oa, oc = Oracle(a), Oracle(c)
    Ha, Hc = oa.integrate_hamiltonian(a.v, a.g), oc.integrate_hamiltonian(c.v, c.g)
    assert np.linalg.norm(Ha - Hc) <= 1e-12 * np.linalg.norm(Ha)
    na, nc = oa.update_density(a.D_values)[0], oc.update_density(c.D_values)[0]
    key = lambda x: np.lexsort((x[:, 2], x[:, 1], x[:, 0]))  # noqa: E731
    assert np.abs(na[key(a.xyz)] - nc[key(c.xyz)]).max() <= 1e-12 * np.abs(na).max()


# --------------------------------------------------------------------------- O4: n, grad n; identities I1-I3
@pytest.mark.parametrize("which", ["cfg1", "toy5", "si"])
def test_trace_identities_tie_density_to_hamiltonian(which, cfg1, toy5):
    if which == "cfg1":
        b = cfg1
    elif which == "toy5":
        b = toy5[0]
    else:
        b = aims_synth.make_config(3, n_rad=10, n_ang=26, keep_atoms=12)
    o = Oracle(b)
    Dd = bsr_to_dense(b, b.D_values)
    n, gn = o.update_density(b.D_values, want_grad=True)
    S = bsr_to_dense(b, o.integrate_hamiltonian(np.ones(b.n_points)))
    Hl = bsr_to_dense(b, o.integrate_hamiltonian(b.v))
    Hg = bsr_to_dense(b, o.integrate_hamiltonian(b.v, b.g))
    i1, r1 = (b.w * n).sum(), (Dd * S).sum()                         # I1: int n = Tr(D S)
    i2, r2 = (b.w * b.v * n).sum(), (Dd * Hl).sum()                  # I2: int v n = Tr(D H_LDA)
    i3, r3 = (b.w * (b.g * gn).sum(0)).sum(), (Dd * (Hg - Hl)).sum()  # I3: int g.grad n = Tr(D H_GGA-term)
    scale = np.abs(Dd).sum() * 0 + max(abs(r1), abs(r2), 1.0)
    assert abs(i1 - r1) < 1e-11 * scale
    assert abs(i2 - r2) < 1e-11 * scale
    assert abs(i3 - r3) < 1e-11 * scale
    assert abs(r3) > 1e-6                                             # the GGA term is really there


def test_density_nonnegative_for_psd_density_matrix(cfg1, cfg1_oracle):
    n, _ = cfg1_oracle.update_density(cfg1.D_values)
    assert n.min() >= -1e-14 * n.max() and n.max() > 0


def test_grad_density_matches_finite_difference_of_density(toy5):
    b, o = toy5
    _, gn = o.update_density(b.D_values, want_grad=True)
    h = 1e-5
    import copy
    for c in range(3):
        nn = []
        for sgn in (+1, -1):
            bb = copy.copy(b)
            bb.xyz = b.xyz.copy()
            bb.xyz[:, c] += sgn * h
            nn.append(Oracle(bb).update_density(b.D_values)[0])
        fd = (nn[0] - nn[1]) / (2 * h)
        # central differences with h = 1e-5 A are meaningless within ~1e-2 A of a nucleus (log-radial shells start
        # at 1e-3 A); compare where the step is small against the distance to every atom
        far = np.linalg.norm(b.xyz[:, None, :] - b.atom_xyz[None, :, :], axis=2).min(1) > 0.1
        assert far.sum() > 500
        assert np.abs(fd - gn[c])[far].max() < 1e-6 * np.abs(gn[:, far]).max()


def test_eval_basis_rows_follow_the_index_list(toy5):
    b, o = toy5
    bi = b.n_batches // 2
    idx, phi, dphi = o.eval_basis(bi, want_grad=True)
    assert phi.shape == (len(idx), b.batch_ptr[bi + 1] - b.batch_ptr[bi]) and dphi.shape == (3,) + phi.shape
    # row of global function i equals the single-function evaluation
    fn_atom = np.repeat(np.arange(b.n_atoms), np.diff(b.atom_fn_ptr))
    k = len(idx) // 2
    a = fn_atom[idx[k]]
    loc = idx[k] - b.atom_fn_ptr[a]
    sp = b.atom_species[a]
    s = b.species_shell_ptr[sp]
    while loc >= 2 * b.shell_l[s] + 1:
        loc -= 2 * b.shell_l[s] + 1
        s += 1
    for p in range(0, phi.shape[1], 7):
        val, gr = o.shell_at_point(a, s, b.xyz[b.batch_ptr[bi] + p])
        assert phi[k, p] == val[loc] and np.array_equal(dphi[:, k, p], gr[loc])
