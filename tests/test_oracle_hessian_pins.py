"""Pins of the oracle's density-Hessian path (oracle/aims_oracle.c, block "Hessian of the density") against
facts fixed by mathematics -- never against the CUDA path:
  * d_c d_e n is the central difference of the (already pinned) grad n evaluated on displaced points;
  * closed form for one s-type Gaussian: n = |phi|^2 = e^{-2 a r^2} / 4 pi, d_c d_e n = n (16 a^2 r_c r_e - 4 a delta_ce);
  * brute force over ALL functions (no batches, no culling, dense D) written in numpy from the oracle's pinned phi, grad phi,
    Hess phi;
  * symmetric D: the result is linear in D and vanishes with it; invariant under re-batching.
"""
import copy
import math

import numpy as np
import pytest

import aims_synth
from aims_synth import bsr_to_dense
from oracle.oracle import Oracle

IC = (0, 1, 2, 0, 0, 1)
IE = (0, 1, 2, 1, 2, 2)


@pytest.fixture(scope="module")
def toy5():
    b = aims_synth.make_config(5, n_rad=14, n_ang=26, max_batch=40, keep_atoms=6)
    return b, Oracle(b)


def test_density_hessian_is_finite_difference_of_density_gradient(toy5):
    b, o = toy5
    Hn = o.density_hessian(b.D_values)
    h = 1e-5
    far = np.linalg.norm(b.xyz[:, None, :] - b.atom_xyz[None, :, :], axis=2).min(1) > 0.1
    assert far.sum() > 500
    scale = np.abs(Hn[:, far]).max()
    for e in range(3):
        g = []
        for sgn in (+1, -1):
            bb = copy.copy(b)
            bb.xyz = b.xyz.copy()
            bb.xyz[:, e] += sgn * h
            g.append(Oracle(bb).update_density(b.D_values, want_grad=True)[1])
        fd = (g[0] - g[1]) / (2 * h)                       # fd[c] = d_e (d_c n)
        for k in range(6):
            for c, ee in ((IC[k], IE[k]), (IE[k], IC[k])):
                if ee == e:
                    assert np.abs(fd[c] - Hn[k])[far].max() < 2e-6 * scale, (k, c, e)


def test_density_hessian_of_one_gaussian_closed_form():
    alpha = 0.9
    b = aims_synth.make_config(1, n_rad=40, n_ang=50, gaussian_s_only=alpha)
    D = np.zeros((3, 3))
    D[0, 0] = 1.0
    Dv = aims_synth.dense_to_bsr(b, D)
    Hn = Oracle(b).density_hessian(Dv)
    r = b.xyz - b.atom_xyz[0]
    r2 = (r ** 2).sum(1)
    inside = (r2 < 4.5 ** 2) & (r2 > 0.05 ** 2)              # the spline table ends at the 5 A cutoff
    n = np.exp(-2 * alpha * r2) / (4 * math.pi)
    for k in range(6):
        ref = n * (16 * alpha ** 2 * r[:, IC[k]] * r[:, IE[k]] - (4 * alpha if IC[k] == IE[k] else 0.0))
        # R is the cubic spline of the tabulated Gaussian (200 knots): R'' is piecewise linear, accurate to ~1e-3
        assert np.abs(Hn[k] - ref)[inside].max() < 2e-3 * np.abs(ref[inside]).max(), k


def test_density_hessian_equals_numpy_brute_force(cfg1, cfg1_oracle, toy5):
    for b, o in ((cfg1, cfg1_oracle), toy5):
        Hn = o.density_hessian(b.D_values)
        Dd = bsr_to_dense(b, b.D_values)
        rng = np.random.default_rng(5)
        pts = rng.choice(b.n_points, 40, replace=False)
        for p in pts:
            phi, gr, he = [], [], []
            for a in range(b.n_atoms):
                sp = b.atom_species[a]
                for s in range(b.species_shell_ptr[sp], b.species_shell_ptr[sp + 1]):
                    v, g, h = o.shell_hess_at_point(a, s, b.xyz[p])
                    phi.append(v), gr.append(g), he.append(h)
            phi, gr, he = np.concatenate(phi), np.vstack(gr), np.vstack(he)
            for k in range(6):
                ref = 2.0 * (he[:, k] @ Dd @ phi + gr[:, IC[k]] @ Dd @ gr[:, IE[k]])
                assert abs(Hn[k, p] - ref) <= 1e-11 * max(np.abs(Hn[:, p]).max(), 1e-12), (p, k)


def test_density_hessian_linear_in_D_and_rebatching():
    a = aims_synth.make_config(1, max_batch=128)
    c = aims_synth.make_config(1, max_batch=37)
    Ha = Oracle(a).density_hessian(a.D_values)
    assert np.abs(Oracle(a).density_hessian(-2.0 * a.D_values) + 2.0 * Ha).max() <= 1e-13 * np.abs(Ha).max()
    # the two batchings order the points differently: compare through the point coordinates
    Hc = Oracle(c).density_hessian(c.D_values)
    ka = np.lexsort(a.xyz.T[::-1])
    kc = np.lexsort(c.xyz.T[::-1])
    assert np.array_equal(a.xyz[ka], c.xyz[kc])
    assert np.abs(Ha[:, ka] - Hc[:, kc]).max() <= 1e-11 * np.abs(Ha).max()
