"""Pins of the oracle's partition of unity (oracle/aims_oracle.c, block "Partition of unity"; Eq. 21-22,
DESIGN.md reading P5) against facts fixed by mathematics -- never against the CUDA path:
  * sum over all owners = 1 at arbitrary points that have a candidate atom, every weight in [0, 1];
  * two atoms: w = 1/2 on the bisecting plane, exactly 1 (0) where mu <= -0.64 (>= 0.64), monotone along the bond;
  * invariant under rigid motions of atoms and points together;
  * used as the integration weight it integrates a Gaussian to its closed form (the grid recipe of DESIGN.md section 4).
"""
import copy
import math

import numpy as np

import aims_synth
from oracle.oracle import Oracle


def _two_atoms(R=2.0):
    b = copy.copy(aims_synth.make_config(1, n_rad=8, n_ang=14))
    b.atom_xyz = np.array([[0.0, 0.0, 0.0], [R, 0.0, 0.0]])
    b.atom_species = b.atom_species[:2].copy()
    return b


def test_weights_sum_to_one_over_owners_and_lie_in_unit_interval():
    b = aims_synth.make_config(5, n_rad=6, n_ang=14, keep_atoms=40)
    o = Oracle(b)
    rng = np.random.default_rng(3)
    pts = b.atom_xyz[rng.integers(0, b.n_atoms, 300)] + rng.normal(0.0, 1.5, (300, 3))
    r_part = 7.0
    tot = np.zeros(len(pts))
    for A in range(b.n_atoms):
        w = o.partition_weights(pts, np.full(len(pts), A), r_part)
        assert w.min() >= 0.0 and w.max() <= 1.0
        tot += w
    assert np.abs(tot - 1.0).max() <= 1e-13


def test_two_atom_limits_midplane_and_monotonicity():
    R = 2.0
    o = Oracle(_two_atoms(R))
    rng = np.random.default_rng(4)
    mid = np.column_stack([np.full(50, R / 2), rng.normal(0, 1, 50), rng.normal(0, 1, 50)])
    assert np.abs(o.partition_weights(mid, np.zeros(50), 10.0) - 0.5).max() <= 1e-15
    x = np.linspace(-1.0, 3.0, 401)
    line = np.column_stack([x, np.zeros_like(x), np.zeros_like(x)])
    w0 = o.partition_weights(line, np.zeros(len(x)), 10.0)
    mu = (np.abs(x) - np.abs(x - R)) / R
    assert np.all(w0[mu <= -0.64] == 1.0) and np.all(w0[mu >= 0.64] == 0.0)
    assert np.all(np.diff(w0[(x > 0) & (x < R)]) <= 1e-16)
    assert np.abs(w0 + o.partition_weights(line, np.ones(len(x)), 10.0) - 1.0).max() <= 1e-15
    # outside the neighbour radius of the owner: not a candidate -> 0
    far = np.array([[30.0, 0.0, 0.0]])
    assert o.partition_weights(far, np.zeros(1), 10.0)[0] == 0.0


def test_invariant_under_rigid_motion():
    b = aims_synth.make_config(5, n_rad=6, n_ang=14, keep_atoms=20)
    rng = np.random.default_rng(5)
    pts = b.atom_xyz[rng.integers(0, b.n_atoms, 200)] + rng.normal(0.0, 1.0, (200, 3))
    own = rng.integers(0, b.n_atoms, 200)
    w = Oracle(b).partition_weights(pts, own, 7.0)
    Qm, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    t = np.array([0.3, -1.2, 2.0])
    b2 = copy.copy(b)
    b2.atom_xyz = np.ascontiguousarray(b.atom_xyz @ Qm.T + t)
    w2 = Oracle(b2).partition_weights(pts @ Qm.T + t, own, 7.0)
    assert np.abs(w - w2).max() <= 1e-12


def test_partitioned_atom_grids_integrate_a_gaussian_to_its_closed_form():
    b = aims_synth.make_config(1, n_rad=40, n_ang=110)
    o = Oracle(b)
    wq = b.w / np.where(aims_synth.partition_weights(b.atom_xyz, b.xyz, b.owner, b.meta["r_part"]) > 0,
                        aims_synth.partition_weights(b.atom_xyz, b.xyz, b.owner, b.meta["r_part"]), 1.0)
    w = wq * o.partition_weights(b.xyz, b.owner, b.meta["r_part"])        # quadrature weight x the ORACLE's partition weight
    c = b.atom_xyz.mean(0)
    for alpha in (0.5, 1.5):
        val = float((w * np.exp(-alpha * ((b.xyz - c) ** 2).sum(1))).sum())
        assert abs(val / (math.pi / alpha) ** 1.5 - 1.0) < 2e-3
