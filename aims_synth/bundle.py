"""make_config(k): assemble one Bundle (see configs.py header; input generation only)."""
from __future__ import annotations

import numpy as np

from .configs import (BASE_SEED, N_KNOTS, R0_KNOT, SPECIES, Bundle, _geometry, _radial_norm, bisect_batches,
                      build_splines, fibonacci_sphere, partition_weights, radial_analytic, radial_grid,
                      smooth_fields)

# (n_rad, n_ang, max_batch) of BASELINE.json configs 1..5
GRID_DEFAULTS = {1: (40, 110, 128), 2: (60, 302, 200), 3: (60, 302, 200), 4: (60, 302, 200), 5: (70, 302, 200)}


def build_bsr(atom_xyz, atom_rc, atom_nfn):
    """Atom-pair block pattern (P13): upper blocks (col >= row) for pairs with |R_A-R_B| < rc(A)+rc(B); block (A,B)
    is row-major [n_fn(A)][ld], ld = n_fn(B) rounded up to even; offsets are multiples of 2 doubles (16 B)."""
    n = len(atom_xyz)
    d = np.linalg.norm(atom_xyz[:, None, :] - atom_xyz[None, :, :], axis=2)
    near = d < (atom_rc[:, None] + atom_rc[None, :])
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    cols, offs, lds = [], [], []
    off = 0
    for a in range(n):
        cb = np.nonzero(near[a, a:])[0] + a
        for b in cb:
            ld = int(atom_nfn[b] + (atom_nfn[b] & 1))
            cols.append(b)
            offs.append(off)
            lds.append(ld)
            off += int(atom_nfn[a]) * ld
        row_ptr[a + 1] = len(cols)
    return (row_ptr, np.array(cols, dtype=np.int32), np.array(offs, dtype=np.int64),
            np.array(lds, dtype=np.int32), int(off))


def bsr_to_dense(bun, values):
    """Expand a block-sparse value array into the full symmetric n_basis x n_basis matrix (bookkeeping only)."""
    nb = bun.n_basis
    M = np.zeros((nb, nb))
    fp = bun.atom_fn_ptr
    for a in range(bun.n_atoms):
        na = fp[a + 1] - fp[a]
        for q in range(bun.row_ptr[a], bun.row_ptr[a + 1]):
            b = bun.col_atom[q]
            nbf = fp[b + 1] - fp[b]
            ld = bun.blk_ld[q]
            blk = values[bun.blk_off[q]: bun.blk_off[q] + na * ld].reshape(na, ld)[:, :nbf]
            M[fp[a]:fp[a + 1], fp[b]:fp[b + 1]] = blk
            if b != a:
                M[fp[b]:fp[b + 1], fp[a]:fp[a + 1]] = blk.T
    return M


def dense_to_bsr(bun, M):
    vals = np.zeros(bun.n_values)
    fp = bun.atom_fn_ptr
    for a in range(bun.n_atoms):
        na = fp[a + 1] - fp[a]
        for q in range(bun.row_ptr[a], bun.row_ptr[a + 1]):
            b = bun.col_atom[q]
            nbf = fp[b + 1] - fp[b]
            ld = bun.blk_ld[q]
            blk = np.zeros((na, ld))
            blk[:, :nbf] = M[fp[a]:fp[a + 1], fp[b]:fp[b + 1]]
            vals[bun.blk_off[q]: bun.blk_off[q] + na * ld] = blk.ravel()
    return vals


def bsr_pad_mask(bun):
    """True at the padding entries (columns >= n_fn(col) of a block), which hold no matrix element."""
    mask = np.zeros(bun.n_values, dtype=bool)
    fp = bun.atom_fn_ptr
    for a in range(bun.n_atoms):
        na = fp[a + 1] - fp[a]
        for q in range(bun.row_ptr[a], bun.row_ptr[a + 1]):
            b = bun.col_atom[q]
            nbf = fp[b + 1] - fp[b]
            ld = bun.blk_ld[q]
            if ld > nbf:
                m = np.zeros((na, ld), dtype=bool)
                m[:, nbf:] = True
                mask[bun.blk_off[q]: bun.blk_off[q] + na * ld] = m.ravel()
    return mask


def make_config(cfg, n_rad=None, n_ang=None, max_batch=None, seed=None, gaussian_s_only=None, keep_atoms=None):
    """Bundle for BASELINE.json config `cfg` (1..5).  n_rad / n_ang / max_batch override the grid (tests use
    coarser grids on the same geometry and basis; config 4 sweeps max_batch).  gaussian_s_only=alpha replaces the
    basis by one pure-Gaussian s shell per atom (exponent alpha, no cutoff factor) for closed-form pins.  keep_atoms=k keeps the first k atoms only (toy clusters for brute-force tests)."""
    d_rad, d_ang, d_mb = GRID_DEFAULTS[cfg]
    n_rad = n_rad or d_rad
    n_ang = n_ang or d_ang
    max_batch = max_batch or d_mb
    if seed is None:
        seed = BASE_SEED + (2 if cfg == 3 else cfg)    # config 3 is config 2's cluster with the GGA fields used
    rng = np.random.default_rng(seed)
    atom_xyz, names = _geometry(cfg, rng)
    if keep_atoms is not None:
        atom_xyz, names = atom_xyz[:keep_atoms], names[:keep_atoms]
    atom_xyz = np.ascontiguousarray(atom_xyz, dtype=np.float64)
    sp_names = sorted(set(names), key=names.index)
    atom_species = np.array([sp_names.index(n) for n in names], dtype=np.int32)

    # ---- species shell tables, one spline per shell
    shell_l, shell_rcut, shell_zeta, shell_norm, ssp = [], [], [], [], [0]
    for sp in sp_names:
        ls, rc = SPECIES[sp]
        if gaussian_s_only is not None:
            ls = [0]
        for l in ls:
            shell_l.append(l)
            shell_rcut.append(rc)
            shell_zeta.append(rng.uniform(0.8, 3.0))
        ssp.append(len(shell_l))
    shell_l = np.array(shell_l, dtype=np.int32)
    shell_rcut = np.array(shell_rcut, dtype=np.float64)
    shell_zeta = np.array(shell_zeta)
    n_shells = len(shell_l)
    rc_max = float(shell_rcut.max())
    log_inc = np.log(rc_max / R0_KNOT) / (N_KNOTS - 1)
    r_knots = R0_KNOT * np.exp(log_inc * np.arange(N_KNOTS))
    tables = np.empty((n_shells, N_KNOTS))
    for s in range(n_shells):
        if gaussian_s_only is not None:
            shell_norm.append(1.0)
            tables[s] = np.exp(-gaussian_s_only * r_knots ** 2)
        else:
            nrm = _radial_norm(shell_l[s], shell_zeta[s], shell_rcut[s])
            shell_norm.append(nrm)
            tables[s] = radial_analytic(r_knots, shell_l[s], shell_zeta[s], shell_rcut[s], nrm)
    spline_coef = build_splines(tables)
    species_shell_ptr = np.array(ssp, dtype=np.int32)
    sp_nfn = np.array([int(np.sum(2 * shell_l[ssp[i]:ssp[i + 1]] + 1)) for i in range(len(sp_names))])
    sp_rc = np.array([float(shell_rcut[ssp[i]:ssp[i + 1]].max()) for i in range(len(sp_names))])
    atom_nfn = sp_nfn[atom_species]
    atom_rc = sp_rc[atom_species]
    atom_fn_ptr = np.concatenate([[0], np.cumsum(atom_nfn)]).astype(np.int64)

    # ---- atom-centred grids: n_rad log-radial shells x n_ang Fibonacci points, atom-major order
    dirs = fibonacci_sphere(n_ang)
    pts, wts, own = [], [], []
    for a in range(len(atom_xyz)):
        r, wr = radial_grid(n_rad, atom_rc[a] + 1.0)
        pts.append((r[:, None, None] * dirs[None, :, :]).reshape(-1, 3) + atom_xyz[a])
        wts.append(np.repeat(wr * (4.0 * np.pi / n_ang), n_ang))
        own.append(np.full(n_rad * n_ang, a, dtype=np.int32))
    xyz = np.ascontiguousarray(np.concatenate(pts))
    w_quad = np.concatenate(wts)
    owner = np.concatenate(own)
    r_part = float(atom_rc.max() + 1.0)
    w = w_quad * partition_weights(atom_xyz, xyz, owner, r_part)

    # ---- batches (points of a batch contiguous, batches depth-first)
    order, batch_ptr = bisect_batches(xyz, max_batch)
    xyz = np.ascontiguousarray(xyz[order])
    w = np.ascontiguousarray(w[order])
    owner = np.ascontiguousarray(owner[order])

    # ---- pattern, fields, density matrix
    row_ptr, col_atom, blk_off, blk_ld, n_values = build_bsr(atom_xyz, atom_rc, atom_nfn)
    na = len(atom_xyz)
    c = rng.uniform(-1.0, -0.1, (na, 3))
    alpha = rng.uniform(0.5, 2.0, (na, 3))
    b = rng.uniform(-0.5, 0.5, na)
    beta = rng.uniform(0.5, 2.0, na)
    v, g = smooth_fields(atom_xyz, xyz, c, alpha, b, beta, want_g=True)

    bun = Bundle(name="config%d" % cfg, seed=int(seed), atom_xyz=atom_xyz, atom_species=atom_species,
                 species_names=sp_names, species_shell_ptr=species_shell_ptr, shell_l=shell_l, shell_rcut=shell_rcut,
                 shell_spline=np.arange(n_shells, dtype=np.int32), r0=R0_KNOT, log_inc=float(log_inc),
                 n_knots=N_KNOTS, spline_coef=spline_coef, shell_zeta=shell_zeta, shell_norm=np.array(shell_norm),
                 xyz=xyz, w=w, batch_ptr=batch_ptr, max_batch_points=int(np.diff(batch_ptr).max(initial=0)),
                 owner=owner, row_ptr=row_ptr, col_atom=col_atom, blk_off=blk_off, blk_ld=blk_ld, n_values=n_values,
                 v=v, g=g, D_values=None, atom_fn_ptr=atom_fn_ptr,
                 meta=dict(cfg=cfg, n_rad=n_rad, n_ang=n_ang, max_batch=max_batch, r_part=r_part,
                           gga=cfg in (1, 3, 4, 5), v_c=c, v_alpha=alpha, g_b=b, g_beta=beta))
    nbas = bun.n_basis
    if cfg == 1:
        C = rng.standard_normal((nbas, 4))
        Dd = C @ C.T                                   # symmetric positive semidefinite
        bun.D_values = dense_to_bsr(bun, Dd)
    else:
        # symmetric uniform[-1,1] * exp(-R_AB / 4 A) on the pattern, zero elsewhere (P21), drawn block by block
        vals = rng.uniform(-1.0, 1.0, n_values)
        rows = np.repeat(np.arange(na), np.diff(row_ptr))
        Rab = np.linalg.norm(atom_xyz[rows] - atom_xyz[col_atom], axis=1)
        vals *= np.repeat(np.exp(-Rab / 4.0), atom_nfn[rows] * blk_ld)
        vals[bsr_pad_mask(bun)] = 0.0
        for a in range(na):                            # diagonal blocks: symmetrise the square
            q = row_ptr[a]                             # first block of a row is the diagonal one (col >= row)
            n, ld = int(atom_nfn[a]), int(blk_ld[q])
            blk = vals[blk_off[q]: blk_off[q] + n * ld].reshape(n, ld)
            blk[:, :n] = 0.5 * (blk[:, :n] + blk[:, :n].T)
        bun.D_values = vals
    return bun


def make_q_values(bun, seed_offset=1000):
    """Stand-in for the energy-weighted density matrix q_ij of PAPER.md Eq. 17 (needs eigenvectors, which this build does not
    have): symmetric uniform[-1,1] * exp(-R_AB / 4 A) on the block pattern, drawn block by block from its own seeded
    stream (bun.seed + seed_offset) exactly like D of configs 2-5 (P21)."""
    rng = np.random.default_rng(bun.seed + seed_offset)
    na = bun.n_atoms
    atom_nfn = np.diff(bun.atom_fn_ptr).astype(np.int64)
    vals = rng.uniform(-1.0, 1.0, bun.n_values)
    rows = np.repeat(np.arange(na), np.diff(bun.row_ptr))
    Rab = np.linalg.norm(bun.atom_xyz[rows] - bun.atom_xyz[bun.col_atom], axis=1)
    vals *= np.repeat(np.exp(-Rab / 4.0), atom_nfn[rows] * bun.blk_ld)
    vals[bsr_pad_mask(bun)] = 0.0
    for a in range(na):
        q = bun.row_ptr[a]
        n, ld = int(atom_nfn[a]), int(bun.blk_ld[q])
        blk = vals[bun.blk_off[q]: bun.blk_off[q] + n * ld].reshape(n, ld)
        blk[:, :n] = 0.5 * (blk[:, :n] + blk[:, :n].T)
    return vals


def make_xi(bun):
    """Stand-in for xi = d f_xc / d tau of a meta-GGA: a smooth positive field derived from the bundle's
    seeded potential, xi_p = 0.3 + v_p^2 (no new random draws, so every bundle variant has one)."""
    return 0.3 + np.asarray(bun.v) ** 2
