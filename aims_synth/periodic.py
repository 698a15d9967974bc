"""Seeded synthetic PERIODIC system (row f3 of SURVEY.md 8(f)): a triclinic cell with two atoms, its
periodic images that reach into the cell (the "N_rs" real-space functions of Eq. 12), atom-centred grids of the cell atoms
whose points are mapped back into the cell at T = (0,0,0) (L113-115), partition weights over all periodic atoms.  Holds none of
the method's arithmetic: the library and the oracle see the images as ordinary atoms -- "the local integrals h^uc_ij can be
computed using the exact same real-space integration code" (L113) -- plus atom_home / atom_T for the Bloch sums.
"""
import numpy as np

from .bundle import bsr_pad_mask, build_bsr
from .configs import (BASE_SEED, N_KNOTS, R0_KNOT, SPECIES, Bundle, _radial_norm, bisect_batches, build_splines, fibonacci_sphere,
                      partition_weights, radial_analytic, radial_grid, smooth_fields)

LATTICE = np.array([[4.2, 0.0, 0.0], [0.6, 4.6, 0.0], [0.3, 0.5, 5.0]])      # rows a1, a2, a3 (Angstrom)
FRAC = np.array([[0.10, 0.15, 0.20], [0.55, 0.60, 0.45]])                    # two atoms, no symmetry between them
SHELLS = [0, 0, 1, 2]                                                        # s, s, p, d: 10 functions per atom


def _images(lat, frac_atoms, reach):
    """(home index, integer translation) of every periodic atom within `reach` of the cell (a superset)."""
    vol = abs(np.linalg.det(lat))
    heights = np.array([vol / np.linalg.norm(np.cross(lat[(i + 1) % 3], lat[(i + 2) % 3])) for i in range(3)])
    delta = reach / heights
    nmax = np.ceil(delta + 1).astype(int)
    out = []
    for n1 in range(-nmax[0], nmax[0] + 1):
        for n2 in range(-nmax[1], nmax[1] + 1):
            for n3 in range(-nmax[2], nmax[2] + 1):
                n = np.array([n1, n2, n3])
                for a, f in enumerate(frac_atoms):
                    ff = f + n
                    if np.all(ff > -delta) and np.all(ff < 1.0 + delta):
                        out.append((a, n1, n2, n3))
    out.sort(key=lambda t: (t[1:] != (0, 0, 0), t[1:], t[0]))                # the cell's own atoms first
    return out


def make_periodic(n_rad=24, n_ang=50, max_batch=100, rcut=4.0, seed=None, gaussian_s_only=None):
    """Bundle of the periodic toy crystal, with extra attributes: lattice [3][3], frac [n_home][3], atom_home [n_atoms] (index of
    the cell atom an atom is an image of), atom_T [n_atoms][3] (its lattice translation, Angstrom), xyz_unwrapped (the grid
    points before they are mapped into the cell, in the batched order).  Atoms 0..n_home-1 are the cell's."""
    seed = BASE_SEED + 77 if seed is None else seed
    rng = np.random.default_rng(seed)
    lat = LATTICE.copy()
    frac = FRAC + rng.uniform(-0.02, 0.02, FRAC.shape)
    return _make(lat, frac, SHELLS, rcut, n_rad, n_ang, max_batch, seed, rng, gaussian_s_only, "periodic")


def make_periodic_si(n_cells=3, n_rad=60, n_ang=302, max_batch=200, seed=None, jitter=0.05):
    """Periodic workload shaped like the paper's main benchmark (a diamond-Si supercell of 54 atoms): n_cells^3
    primitive fcc cells of the diamond structure (a = 5.43 Angstrom, two atoms per primitive cell: 54 atoms for n_cells = 3),
    positions jittered by +-jitter Angstrom from the seed, the basis and grid of BASELINE.json's config 2/3 (13 functions per atom:
    s, s, p, p, d; cutoff 6 Angstrom; 60 x 302 points per atom; batches of <= 200 points), GGA fields.  Stands in for the paper's
    FHI-aims "tight" silicon run, which is not in this container."""
    seed = BASE_SEED + 54 if seed is None else seed
    rng = np.random.default_rng(seed)
    a = 5.43
    prim = 0.5 * a * np.array([[0.0, 1.0, 1.0], [1.0, 0.0, 1.0], [1.0, 1.0, 0.0]])
    lat = n_cells * prim
    cells = np.array([[i, j, k] for i in range(n_cells) for j in range(n_cells) for k in range(n_cells)], dtype=np.float64)
    frac = np.concatenate([(cells + f) / n_cells for f in (np.zeros(3), np.full(3, 0.25))])
    frac = frac + (rng.uniform(-jitter, jitter, frac.shape) @ np.linalg.inv(lat))
    frac = frac - np.floor(frac)
    ls, rcut = SPECIES["Si"]
    return _make(lat, frac, list(ls), rcut, n_rad, n_ang, max_batch, seed, rng, None, "periodic_si%d" % len(frac))


def _make(lat, frac, shells, rcut, n_rad, n_ang, max_batch, seed, rng, gaussian_s_only, name):
    n_home = len(frac)
    img = _images(lat, frac, rcut)
    atom_home = np.array([t[0] for t in img], dtype=np.int32)
    atom_n = np.array([t[1:] for t in img], dtype=np.int64)
    atom_T = np.ascontiguousarray(atom_n @ lat, dtype=np.float64)
    atom_xyz = np.ascontiguousarray(frac[atom_home] @ lat + atom_T)
    na = len(atom_xyz)
    assert np.all(atom_n[:n_home] == 0) and np.array_equal(atom_home[:n_home], np.arange(n_home))

    ls = [0] if gaussian_s_only is not None else shells
    shell_l = np.array(ls, dtype=np.int32)
    n_shells = len(ls)
    shell_rcut = np.full(n_shells, rcut)
    shell_zeta = rng.uniform(0.8, 3.0, n_shells)
    log_inc = np.log(rcut / R0_KNOT) / (N_KNOTS - 1)
    r_knots = R0_KNOT * np.exp(log_inc * np.arange(N_KNOTS))
    tables, shell_norm = np.empty((n_shells, N_KNOTS)), []
    for s in range(n_shells):
        if gaussian_s_only is not None:
            shell_norm.append(1.0)
            tables[s] = np.exp(-gaussian_s_only * r_knots ** 2)
        else:
            shell_norm.append(_radial_norm(shell_l[s], shell_zeta[s], rcut))
            tables[s] = radial_analytic(r_knots, shell_l[s], shell_zeta[s], rcut, shell_norm[-1])
    spline_coef = build_splines(tables)
    nfn = int(np.sum(2 * shell_l + 1))
    atom_nfn = np.full(na, nfn)
    atom_rc = np.full(na, rcut)
    atom_fn_ptr = np.concatenate([[0], np.cumsum(atom_nfn)]).astype(np.int64)

    # grids of the cell atoms; partition over ALL periodic atoms near them; then map the points into the cell
    r_part = rcut + 1.0
    part = _images(lat, frac, 2.0 * r_part + 1.0)
    part_xyz = np.array([frac[t[0]] + np.array(t[1:]) for t in part]) @ lat
    part_home_idx = [k for k, t in enumerate(part) if t[1:] == (0, 0, 0)]
    dirs = fibonacci_sphere(n_ang)
    pts, wts, own = [], [], []
    for a in range(n_home):
        r, wr = radial_grid(n_rad, r_part)
        pts.append((r[:, None, None] * dirs[None, :, :]).reshape(-1, 3) + atom_xyz[a])
        wts.append(np.repeat(wr * (4.0 * np.pi / n_ang), n_ang))
        own.append(np.full(n_rad * n_ang, part_home_idx[a], dtype=np.int32))
    xyz = np.concatenate(pts)
    w = np.concatenate(wts) * partition_weights(part_xyz, xyz, np.concatenate(own), r_part)
    xyz_unwrapped = xyz
    fr = xyz @ np.linalg.inv(lat)
    xyz = np.ascontiguousarray((fr - np.floor(fr)) @ lat)                     # L113-115: back into the cell at T = 0
    owner = np.concatenate([np.full(n_rad * n_ang, a, dtype=np.int32) for a in range(n_home)])

    order, batch_ptr = bisect_batches(xyz, max_batch)
    xyz, w, owner = np.ascontiguousarray(xyz[order]), np.ascontiguousarray(w[order]), np.ascontiguousarray(owner[order])
    xyz_unwrapped = np.ascontiguousarray(xyz_unwrapped[order])

    row_ptr, col_atom, blk_off, blk_ld, n_values = build_bsr(atom_xyz, atom_rc, atom_nfn)
    # periodic smooth fields: the same Gaussians on every image of a cell atom
    c = rng.uniform(-1.0, -0.1, (n_home, 3))[[t[0] for t in part]]
    alpha = rng.uniform(0.5, 2.0, (n_home, 3))[[t[0] for t in part]]
    bb = rng.uniform(-0.5, 0.5, n_home)[[t[0] for t in part]]
    beta = rng.uniform(0.5, 2.0, n_home)[[t[0] for t in part]]
    v, g = smooth_fields(part_xyz, xyz, c, alpha, bb, beta, want_g=True)

    bun = Bundle(name=name, seed=int(seed), atom_xyz=atom_xyz, atom_species=np.zeros(na, dtype=np.int32),
                 species_names=["P"], species_shell_ptr=np.array([0, n_shells], dtype=np.int32), shell_l=shell_l,
                 shell_rcut=shell_rcut, shell_spline=np.arange(n_shells, dtype=np.int32), r0=R0_KNOT, log_inc=float(log_inc),
                 n_knots=N_KNOTS, spline_coef=spline_coef, shell_zeta=shell_zeta, shell_norm=np.array(shell_norm),
                 xyz=xyz, w=w, batch_ptr=batch_ptr, max_batch_points=int(np.diff(batch_ptr).max(initial=0)), owner=owner,
                 row_ptr=row_ptr, col_atom=col_atom, blk_off=blk_off, blk_ld=blk_ld, n_values=n_values, v=v, g=g,
                 D_values=None, atom_fn_ptr=atom_fn_ptr,
                 meta=dict(cfg="periodic", n_rad=n_rad, n_ang=n_ang, max_batch=max_batch, r_part=r_part, gga=True))
    vals = rng.uniform(-1.0, 1.0, n_values)      # symmetric random D on the pattern (parity does not need translational invariance)
    rows = np.repeat(np.arange(na), np.diff(row_ptr))
    vals *= np.repeat(np.exp(-np.linalg.norm(atom_xyz[rows] - atom_xyz[col_atom], axis=1) / 4.0), atom_nfn[rows] * blk_ld)
    vals[bsr_pad_mask(bun)] = 0.0
    for a in range(na):
        q = row_ptr[a]
        blk = vals[blk_off[q]: blk_off[q] + nfn * int(blk_ld[q])].reshape(nfn, int(blk_ld[q]))
        blk[:, :nfn] = 0.5 * (blk[:, :nfn] + blk[:, :nfn].T)
    bun.D_values = vals
    bun.lattice, bun.atom_home, bun.atom_T, bun.n_home = lat, atom_home, atom_T, n_home
    bun.frac, bun.atom_n, bun.xyz_unwrapped, bun.rcut = frac, atom_n.astype(np.int32), xyz_unwrapped, float(rcut)
    return bun
