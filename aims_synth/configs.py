"""Seeded synthetic inputs shaped like the workloads of arXiv:1912.06636 (BASELINE.json configs 1-5).

INPUT GENERATION ONLY: geometry, species shell tables, radial tables -> spline coefficients, atom-centred
grids with partition weights, cut-plane batches, the atom-pair block-sparse pattern, v(r), g(r) and D.
None of the method's arithmetic (basis evaluation, culling, contractions) lives here; both the CPU oracle
(oracle/) and the CUDA path (paper_1912_06636_b200/) consume exactly these arrays.  The recipe is stated in
DESIGN.md section "Input recipe"; readings P3-P5, P8, P9, P12, P13, P17-P19, P21 of SURVEY.md section 8(c).

They stand in for the paper's FHI-aims workloads (54-atom Si, the 103-compound set, the 375-atom Bi2Se3 slab;
PAPER.md L450-451, L535), whose structures, species files and Lebedev tables are not available here.
"""
from __future__ import annotations

import ctypes
import math
from dataclasses import dataclass, field

import numpy as np

from . import _build

BASE_SEED = 19120663

# l of each radial shell, and the cutoff radius (Angstrom) shared by the species' shells
SPECIES = {
    "O": ([0, 0, 1], 5.0),
    "H": ([0, 0], 5.0),
    "Si": ([0, 0, 1, 1, 2], 6.0),
    "A": ([0, 0, 1, 1, 2, 2], 5.0),
    "B": ([0, 0, 1, 1, 1, 2, 2, 3], 7.0),
    "Bi": ([0] * 3 + [1] * 3 + [2] * 4 + [3], 6.0),
    "Se": ([0] * 4 + [1] * 2 + [2] * 3 + [3], 6.0),
}

R0_KNOT = 5.0e-4      # first spline knot (Angstrom)
N_KNOTS = 200         # BASELINE config 1: "tabulated on a 200-point log grid"
R_MIN_GRID = 1.0e-3   # innermost radial shell of an atom grid
CUT_WIDTH = 2.0       # smooth cutoff acts on the last 2 Angstrom (P9)
R_FIELD = 8.0         # neighbour radius for the synthetic v, g fields


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


@dataclass
class Bundle:
    """All inputs of one configuration (numpy arrays, C-contiguous, the dtypes of include/aims_gpu.h)."""
    name: str
    seed: int
    # basis (aims_basis_desc)
    atom_xyz: np.ndarray
    atom_species: np.ndarray
    species_names: list
    species_shell_ptr: np.ndarray
    shell_l: np.ndarray
    shell_rcut: np.ndarray
    shell_spline: np.ndarray
    r0: float
    log_inc: float
    n_knots: int
    spline_coef: np.ndarray
    shell_zeta: np.ndarray
    shell_norm: np.ndarray
    # grid (aims_grid_desc)
    xyz: np.ndarray
    w: np.ndarray
    batch_ptr: np.ndarray
    max_batch_points: int
    owner: np.ndarray
    # block-sparse pattern (aims_bsr_desc)
    row_ptr: np.ndarray
    col_atom: np.ndarray
    blk_off: np.ndarray
    blk_ld: np.ndarray
    n_values: int
    # fields
    v: np.ndarray
    g: np.ndarray
    D_values: np.ndarray
    # derived index helpers (plain bookkeeping)
    atom_fn_ptr: np.ndarray = field(default=None)
    meta: dict = field(default_factory=dict)

    @property
    def n_atoms(self):
        return int(self.atom_xyz.shape[0])

    @property
    def n_points(self):
        return int(self.xyz.shape[0])

    @property
    def n_batches(self):
        return int(self.batch_ptr.shape[0] - 1)

    @property
    def n_basis(self):
        return int(self.atom_fn_ptr[-1])


# ----------------------------------------------------------------------------- geometry
def _geometry(cfg, rng):
    if cfg == 1:
        xyz = np.array([[0.0, 0.0, 0.0], [0.96, 0.0, 0.0], [-0.24, 0.93, 0.0]])
        return xyz, ["O", "H", "H"]
    if cfg in (2, 3):
        a = 5.43
        frac = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0],
                         [.25, .25, .25], [.25, .75, .75], [.75, .25, .75], [.75, .75, .25]])
        cells = np.array([[i, j, k] for i in range(2) for j in range(2) for k in range(2)], dtype=float)
        xyz = (cells[:, None, :] + frac[None, :, :]).reshape(-1, 3) * a
        xyz = xyz + rng.uniform(-0.05, 0.05, xyz.shape)
        return xyz, ["Si"] * len(xyz)
    if cfg == 4:
        p = 2.8
        sites, names = [], []
        for i in range(10):
            for j in range(10):
                for k in range(2):
                    sites.append([i * p, j * p, k * p])
                    names.append("A" if (i + j + k) % 2 == 0 else "B")
        xyz = np.array(sites) + rng.uniform(-0.05, 0.05, (len(sites), 3))
        return xyz, names
    if cfg == 5:
        a = 4.14
        a1 = np.array([a, 0.0, 0.0])
        a2 = np.array([a / 2, a * math.sqrt(3) / 2, 0.0])
        z_layer = [0.0, 1.6, 3.5, 5.4, 7.0]
        sp_layer = ["Se", "Bi", "Se", "Bi", "Se"]
        shift_layer = [0, 1, 2, 0, 1]
        sites, names = [], []
        for q in range(3):                       # three quintuple layers -> 375 atoms (P17)
            for lay in range(5):
                s = ((shift_layer[lay] + 2 * q) % 3) / 3.0
                for i in range(5):
                    for j in range(5):
                        r = (i + s) * a1 + (j + s) * a2
                        sites.append([r[0], r[1], z_layer[lay] + 10.0 * q])
                        names.append(sp_layer[lay])
        xyz = np.array(sites) + rng.uniform(-0.05, 0.05, (len(sites), 3))
        return xyz, names
    raise ValueError("config must be 1..5")


# ----------------------------------------------------------------------------- radial tables and splines
def cutoff_fn(r, rcut):
    """1 for r <= rcut-2, quintic smoothstep 1-10x^3+15x^4-6x^5 on the last 2 A, 0 beyond (P9)."""
    x = np.clip((r - (rcut - CUT_WIDTH)) / CUT_WIDTH, 0.0, 1.0)
    return 1.0 - x ** 3 * (10.0 - 15.0 * x + 6.0 * x * x)


def radial_analytic(r, l, zeta, rcut, norm=1.0):
    return norm * r ** l * np.exp(-zeta * r) * cutoff_fn(r, rcut)


def _radial_norm(l, zeta, rcut):
    r = np.linspace(0.0, rcut, 20001)
    f = radial_analytic(r, l, zeta, rcut) ** 2 * r * r
    return 1.0 / math.sqrt(np.trapezoid(f, r))


def build_splines(tables):
    """Natural cubic spline in the knot-index coordinate t (knots at t = 0,1,...): coef[s][k] = (a,b,c,d) with
    R(t) = a + b x + c x^2 + d x^3, x = t - k (P8).  scipy's CubicSpline is the construction; the coefficient
    table it returns is, from here on, the definition of R for both sides."""
    from scipy.interpolate import CubicSpline
    n_spl, n_k = tables.shape
    t = np.arange(n_k, dtype=float)
    coef = np.empty((n_spl, n_k - 1, 4))
    for s in range(n_spl):
        cs = CubicSpline(t, tables[s], bc_type="natural")
        coef[s, :, 0] = cs.c[3]
        coef[s, :, 1] = cs.c[2]
        coef[s, :, 2] = cs.c[1]
        coef[s, :, 3] = cs.c[0]
    return np.ascontiguousarray(coef)


# ----------------------------------------------------------------------------- grids
def fibonacci_sphere(n):
    """n equal-weight points (P4): z_i = 1-(2i+1)/n, phi_i = i*pi*(3-sqrt 5)."""
    i = np.arange(n, dtype=float)
    z = 1.0 - (2.0 * i + 1.0) / n
    ph = i * math.pi * (3.0 - math.sqrt(5.0))
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(ph), s * np.sin(ph), z], axis=1)


def radial_grid(n_rad, r_max):
    """r_s = r_min exp(alpha s); weight alpha r_s^3 with halved ends (trapezoid in s) (P3)."""
    alpha = math.log(r_max / R_MIN_GRID) / (n_rad - 1)
    r = R_MIN_GRID * np.exp(alpha * np.arange(n_rad))
    wr = alpha * r ** 3
    wr[0] *= 0.5
    wr[-1] *= 0.5
    return r, wr


def partition_weights(atom_xyz, xyz, owner, r_part):
    """w_owner(r) of the neighbour-restricted Stratmann partition (see _heavy.c)."""
    atom_xyz = np.ascontiguousarray(atom_xyz, dtype=np.float64)
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    owner = np.ascontiguousarray(owner, dtype=np.int32)
    out = np.empty(len(xyz))
    rc = _build.lib().synth_partition_weights(len(atom_xyz), _dp(atom_xyz), len(xyz), _dp(xyz),
                                              owner.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                                              float(r_part), _dp(out))
    if rc < 0:
        raise RuntimeError("partition_weights: candidate list overflow")
    return out


def bisect_batches(xyz, max_pts):
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    n = len(xyz)
    order = np.empty(n, dtype=np.int64)
    cap = 2 * ((n + max_pts - 1) // max_pts) + 2
    ptr = np.empty(cap, dtype=np.int64)
    lp = ctypes.POINTER(ctypes.c_int64)
    nb = _build.lib().synth_bisect(n, _dp(xyz), int(max_pts), order.ctypes.data_as(lp), ptr.ctypes.data_as(lp))
    return order, np.ascontiguousarray(ptr[: nb + 1])


def smooth_fields(atom_xyz, xyz, c, alpha, b, beta, want_g=True):
    atom_xyz = np.ascontiguousarray(atom_xyz, dtype=np.float64)
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    n = len(xyz)
    v = np.empty(n)
    g = np.empty((3, n)) if want_g else None
    rc = _build.lib().synth_fields(len(atom_xyz), _dp(atom_xyz), c.shape[1], _dp(c), _dp(alpha), _dp(b), _dp(beta),
                                   R_FIELD, n, _dp(xyz), _dp(v), _dp(g) if want_g else None)
    if rc < 0:
        raise RuntimeError("smooth_fields: candidate list overflow")
    return v, g
