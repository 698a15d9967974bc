"""Plain statements of the two geometric steps of the periodic real-space path (Eq. 11-12) -- the oracle of
aims_gpu_periodic_images and aims_gpu_wrap_points.  TEST INFRASTRUCTURE, NOT THE PRODUCT; imports nothing from
paper_1912_06636_b200 and nothing from the input generator.

The paper: h^uc of Eq. 12 runs over "all N_rs basis functions phi_I that are non-zero on the unit cell", centred in the cell or
in its periodic images (L109-113), and "each integration point r is mapped back to its periodic image within the unit cell at
T = (0,0,0)" (L113-115); it states neither how the images are enumerated nor how a point is mapped.  DESIGN.md reading P23:

  images   lattice rows a_1, a_2, a_3; h_i = V / |a_j x a_k| is the height of the cell along the i-th reciprocal direction,
           delta_i = reach / h_i.  The periodic atom (a, n) -- cell atom a with fractional coordinates f_a, translated by the
           integer vector n -- is KEPT iff  -delta_i < f_a,i + n_i < 1 + delta_i  for i = 1, 2, 3  (a parallelepiped that contains
           every point within `reach` of the cell: a superset of the atoms whose functions reach into the cell; the culling of
           S1a drops the rest per batch).  Order: the cell's own atoms (n = 0) first, then ascending (n_1, n_2, n_3, a).
  wrap     f = r A^-1 with A^-1 from the cofactor formula, f <- f - floor(f), and f <- 0 where that difference rounds to 1
           (a tiny negative f: 1 - 1e-20 is not a double; the face f = 1 is the face f = 0 of the next cell, so the point is
           put on f = 0 and the promised range [0, 1) holds), r <- f A; every product and sum separately rounded, sums left to
           right -- one result is correct to the last bit.
Pins (tests/test_oracle_periodic_pins.py): every atom within `reach` of a dense sample of cell points is in the list, no atom
twice, brute force over a large integer box; wrapped points differ from the originals by an integer lattice vector, have
fractional coordinates in [0, 1), wrapping is idempotent; and both reproduce the atoms / points of the seeded periodic bundle
whose Bloch sums are pinned by closed-form Gaussian lattice sums.
"""
import numpy as np


def cell_heights(lat):
    lat = np.asarray(lat, dtype=np.float64)
    vol = abs(float(np.dot(lat[0], np.cross(lat[1], lat[2]))))
    return np.array([vol / np.linalg.norm(np.cross(lat[(i + 1) % 3], lat[(i + 2) % 3])) for i in range(3)])


def periodic_images(lat, frac, reach):
    """(atom_home [n], atom_n [n][3]) of reading P23."""
    lat = np.asarray(lat, dtype=np.float64)
    frac = np.asarray(frac, dtype=np.float64).reshape(-1, 3)
    delta = reach / cell_heights(lat)
    nmax = np.ceil(delta + 1.0).astype(int)
    out = []
    for n1 in range(-nmax[0], nmax[0] + 1):
        for n2 in range(-nmax[1], nmax[1] + 1):
            for n3 in range(-nmax[2], nmax[2] + 1):
                for a in range(len(frac)):
                    ff = frac[a] + np.array([n1, n2, n3], dtype=np.float64)
                    if np.all(ff > -delta) and np.all(ff < 1.0 + delta):
                        out.append((0 if (n1, n2, n3) == (0, 0, 0) else 1, n1, n2, n3, a))
    out.sort()
    home = np.array([t[4] for t in out], dtype=np.int32)
    n = np.array([t[1:4] for t in out], dtype=np.int32).reshape(-1, 3)
    return home, n


def inverse_lattice(lat):
    """A^-1 by cofactors: inv[i][j] = cof[j][i] / det, det expanded along the first row, every operation separately rounded."""
    a = np.asarray(lat, dtype=np.float64)
    cof = np.empty((3, 3))
    for i in range(3):
        for j in range(3):
            r0, r1 = (i + 1) % 3, (i + 2) % 3
            c0, c1 = (j + 1) % 3, (j + 2) % 3
            cof[i, j] = a[r0, c0] * a[r1, c1] - a[r0, c1] * a[r1, c0]        # cyclic indices: the sign is already right
    det = (a[0, 0] * cof[0, 0] + a[0, 1] * cof[0, 1]) + a[0, 2] * cof[0, 2]
    return cof.T / det


def wrap_points(lat, xyz):
    """Points mapped into the cell at T = 0 (reading P23); plain numpy element-wise arithmetic (no FMA contraction)."""
    a = np.asarray(lat, dtype=np.float64)
    inv = inverse_lattice(a)
    r = np.asarray(xyz, dtype=np.float64).reshape(-1, 3)
    f = np.empty_like(r)
    for j in range(3):
        f[:, j] = (r[:, 0] * inv[0, j] + r[:, 1] * inv[1, j]) + r[:, 2] * inv[2, j]
    f = f - np.floor(f)
    f[f >= 1.0] = 0.0                          # -tiny - floor(-tiny) rounds to 1.0: the same face as 0.0, and [0, 1) is the promise
    out = np.empty_like(r)
    for j in range(3):
        out[:, j] = (f[:, 0] * a[0, j] + f[:, 1] * a[1, j]) + f[:, 2] * a[2, j]
    return out
