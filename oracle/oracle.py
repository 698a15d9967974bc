"""ctypes front end of oracle/aims_oracle.c -- the plain FP64 CPU oracle.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this.  It imports nothing from paper_1912_06636_b200 (the CUDA path).
Argument marshalling only; every formula lives in aims_oracle.c, each with its PAPER.md citation.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "aims_oracle.c")
_LIB = os.path.join(_HERE, "libaims_oracle.so")
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int32)
_lp = ctypes.POINTER(ctypes.c_int64)


class _System(ctypes.Structure):
    _fields_ = [("n_atoms", ctypes.c_int32), ("n_species", ctypes.c_int32), ("n_shells", ctypes.c_int32),
                ("n_splines", ctypes.c_int32), ("n_knots", ctypes.c_int32),
                ("atom_xyz", _dp), ("atom_species", _ip), ("species_shell_ptr", _ip), ("shell_l", _ip),
                ("shell_rcut", _dp), ("shell_spline", _ip), ("r0", ctypes.c_double), ("log_inc", ctypes.c_double),
                ("spline_coef", _dp),
                ("n_points", ctypes.c_int64), ("n_batches", ctypes.c_int32),
                ("xyz", _dp), ("w", _dp), ("batch_ptr", _lp),
                ("row_ptr", _lp), ("col_atom", _ip), ("blk_off", _lp), ("blk_ld", _ip), ("n_values", ctypes.c_int64)]


def build(force=False):
    """gcc -O2 -fopenmp -ffp-contract=off (no FMA contraction: the culling predicate of reading P6 needs separately
    rounded multiplies and adds)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        sp = ctypes.POINTER(_System)
        L.orc_solid_harmonics.argtypes = [ctypes.c_int, _dp, _dp, _dp]
        L.orc_radial.argtypes = [sp, ctypes.c_int, ctypes.c_double, _dp, _dp]
        L.orc_shell_at_point.argtypes = [sp, ctypes.c_int, ctypes.c_int, _dp, _dp, _dp]
        L.orc_atom_fn_ptr.argtypes = [sp, _lp]
        L.orc_batch_nnz.restype = ctypes.c_int
        L.orc_batch_nnz.argtypes = [sp, ctypes.c_int, _ip, _ip, _ip, _ip]
        L.orc_eval_basis.argtypes = [sp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _ip, _ip, _ip, _dp, _dp]
        L.orc_integrate_hamiltonian.argtypes = [sp, ctypes.c_int, _ip, _dp, _dp, _dp]
        L.orc_update_density.argtypes = [sp, ctypes.c_int, _ip, _dp, _dp, _dp]
        L.orc_brute.argtypes = [sp, _dp, _dp, _dp, _dp, _dp, _dp]
        L.orc_solid_harmonics_hess.argtypes = [ctypes.c_int, _dp, _dp]
        L.orc_radial2.argtypes = [sp, ctypes.c_int, ctypes.c_double, _dp, _dp, _dp]
        L.orc_shell_hess_at_point.argtypes = [sp, ctypes.c_int, ctypes.c_int, _dp, _dp, _dp, _dp]
        L.orc_pulay_forces.argtypes = [sp, ctypes.c_int, _ip, _dp, _dp, _dp, _dp, ctypes.c_int, _dp]
        L.orc_brute_forces.argtypes = [sp, _dp, _dp, _dp, _dp, ctypes.c_int, _dp]
        L.orc_pulay_stress.argtypes = [sp, ctypes.c_int, _ip, _dp, _dp, _dp, _dp, ctypes.c_int, ctypes.c_double, _dp]
        L.orc_brute_stress.argtypes = [sp, _dp, _dp, _dp, _dp, ctypes.c_double, _dp]
        L.orc_brute_stress_ks.argtypes = [sp, _dp, _dp, _dp, _dp, ctypes.c_int, ctypes.c_double, _dp]
        L.orc_integrate_hamiltonian_ks.argtypes = [sp, ctypes.c_int, _ip, _dp, _dp, ctypes.c_int, _dp]
        L.orc_brute_kinetic.argtypes = [sp, _dp, _dp]
        L.orc_density_hessian.argtypes = [sp, ctypes.c_int, _ip, _dp, _dp]
        L.orc_partition_weights.argtypes = [sp, ctypes.c_int64, _dp, _ip, ctypes.c_double, _dp]
        L.orc_tau_matrix.argtypes = [sp, ctypes.c_int, _ip, _dp, _dp]
        L.orc_bloch_fold.argtypes = [sp, _dp, _ip, _dp, ctypes.c_int, _dp, _dp, _dp]
        _lib = L
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def _l(a):
    return a.ctypes.data_as(_lp)


def num_threads():
    L = _load()
    L.orc_num_threads.restype = ctypes.c_int
    return int(L.orc_num_threads())


def solid_harmonics(l, u, want_grad=False):
    """Y[2l+1] (and grad S_lm [2l+1][3]) at the 3-vector u (O1, reading P10)."""
    u = np.ascontiguousarray(u, dtype=np.float64)
    Y = np.zeros(2 * l + 1)
    G = np.zeros((2 * l + 1, 3)) if want_grad else None
    _load().orc_solid_harmonics(int(l), _d(u), _d(Y), _d(G))
    return (Y, G) if want_grad else Y


def solid_harmonics_hess(l, u):
    """Second derivatives of S_lm at u: [2l+1][6] = (xx, yy, zz, xy, xz, yz)."""
    u = np.ascontiguousarray(u, dtype=np.float64)
    H = np.zeros((2 * l + 1, 6))
    _load().orc_solid_harmonics_hess(int(l), _d(u), _d(H))
    return H


class Oracle:
    """Holds one input bundle (arrays of aims_synth.Bundle, or anything with the same attribute names)."""

    def __init__(self, bun):
        self.L = _load()
        f64 = lambda a: np.ascontiguousarray(a, dtype=np.float64)  # noqa: E731
        i32 = lambda a: np.ascontiguousarray(a, dtype=np.int32)    # noqa: E731
        i64 = lambda a: np.ascontiguousarray(a, dtype=np.int64)    # noqa: E731
        self.keep = dict(atom_xyz=f64(bun.atom_xyz), atom_species=i32(bun.atom_species),
                         species_shell_ptr=i32(bun.species_shell_ptr), shell_l=i32(bun.shell_l),
                         shell_rcut=f64(bun.shell_rcut), shell_spline=i32(bun.shell_spline),
                         spline_coef=f64(bun.spline_coef), xyz=f64(bun.xyz), w=f64(bun.w), batch_ptr=i64(bun.batch_ptr),
                         row_ptr=i64(bun.row_ptr), col_atom=i32(bun.col_atom), blk_off=i64(bun.blk_off),
                         blk_ld=i32(bun.blk_ld))
        k = self.keep
        self.n_points = int(k["xyz"].shape[0])
        self.n_batches = int(k["batch_ptr"].shape[0] - 1)
        self.n_values = int(bun.n_values)
        self.sys = _System(int(k["atom_xyz"].shape[0]), int(k["species_shell_ptr"].shape[0] - 1),
                           int(k["shell_l"].shape[0]), int(k["spline_coef"].shape[0]), int(bun.n_knots),
                           _d(k["atom_xyz"]), _i(k["atom_species"]), _i(k["species_shell_ptr"]), _i(k["shell_l"]),
                           _d(k["shell_rcut"]), _i(k["shell_spline"]), float(bun.r0), float(bun.log_inc),
                           _d(k["spline_coef"]), self.n_points, self.n_batches, _d(k["xyz"]), _d(k["w"]),
                           _l(k["batch_ptr"]), _l(k["row_ptr"]), _i(k["col_atom"]), _l(k["blk_off"]), _i(k["blk_ld"]),
                           self.n_values)
        fp = np.zeros(self.sys.n_atoms + 1, dtype=np.int64)
        self.L.orc_atom_fn_ptr(ctypes.byref(self.sys), _l(fp))
        self.atom_fn_ptr = fp
        self.n_basis = int(fp[-1])

    # ---- O1 pieces
    def radial(self, spline, d):
        R, dR = ctypes.c_double(), ctypes.c_double()
        self.L.orc_radial(ctypes.byref(self.sys), int(spline), float(d), ctypes.byref(R), ctypes.byref(dR))
        return R.value, dR.value

    def shell_at_point(self, atom, shell, r, want_grad=True):
        l = int(self.keep["shell_l"][shell])
        r = np.ascontiguousarray(r, dtype=np.float64)
        phi = np.zeros(2 * l + 1)
        gr = np.zeros((2 * l + 1, 3)) if want_grad else None
        self.L.orc_shell_at_point(ctypes.byref(self.sys), int(atom), int(shell), _d(r), _d(phi), _d(gr))
        return (phi, gr) if want_grad else phi

    # ---- O2
    def batch_nnz(self, b):
        """(fn_index, fn_atom, fn_shell, fn_m) of batch b, ascending global index."""
        cap = max(self.n_basis, 1)
        idx, fa, fs, fm = (np.zeros(cap, dtype=np.int32) for _ in range(4))
        n = self.L.orc_batch_nnz(ctypes.byref(self.sys), int(b), _i(idx), _i(fa), _i(fs), _i(fm))
        return idx[:n].copy(), fa[:n].copy(), fs[:n].copy(), fm[:n].copy()

    # ---- O1 on a batch
    def eval_basis(self, b, want_grad=False):
        """(fn_index, phi[nnz][n_p], dphi[3][nnz][n_p] or None)"""
        idx, fa, fs, fm = self.batch_nnz(b)
        bp = self.keep["batch_ptr"]
        npts = int(bp[b + 1] - bp[b])
        nnz = len(idx)
        phi = np.zeros((nnz, npts))
        dphi = np.zeros((3, nnz, npts)) if want_grad else None
        if nnz and npts:
            self.L.orc_eval_basis(ctypes.byref(self.sys), int(b), int(bool(want_grad)), nnz, _i(fa), _i(fs), _i(fm),
                                  _d(phi), _d(dphi))
        return idx, phi, dphi

    def _sel(self, batches):
        if batches is None:
            batches = np.arange(self.n_batches)
        return np.ascontiguousarray(batches, dtype=np.int32)

    # ---- O3
    def integrate_hamiltonian(self, v, g=None, batches=None, H_values=None):
        sel = self._sel(batches)
        v = np.ascontiguousarray(v, dtype=np.float64)
        g = None if g is None else np.ascontiguousarray(g, dtype=np.float64)
        H = np.zeros(self.n_values) if H_values is None else H_values
        self.L.orc_integrate_hamiltonian(ctypes.byref(self.sys), len(sel), _i(sel), _d(v), _d(g), _d(H))
        return H

    def integrate_hamiltonian_ks(self, v, g=None, kinetic=True, batches=None):
        """H with (h phi) = -1/2 lap phi + v phi symmetrised as in Fig. 6a (DSYR2K, alpha = 1/2) plus the GGA term."""
        sel = self._sel(batches)
        v = np.ascontiguousarray(v, dtype=np.float64)
        g = None if g is None else np.ascontiguousarray(g, dtype=np.float64)
        H = np.zeros(self.n_values)
        self.L.orc_integrate_hamiltonian_ks(ctypes.byref(self.sys), len(sel), _i(sel), _d(v), _d(g), int(bool(kinetic)), _d(H))
        return H

    def tau_matrix(self, xi, batches=None, H_values=None):
        """H_values += 1/2 sum_p w xi grad phi_i . grad phi_j (meta-GGA tau matrix, reading P1c)."""
        sel = self._sel(batches)
        xi = np.ascontiguousarray(xi, dtype=np.float64)
        H = np.zeros(self.n_values) if H_values is None else H_values
        self.L.orc_tau_matrix(ctypes.byref(self.sys), len(sel), _i(sel), _d(xi), _d(H))
        return H

    def brute_kinetic(self, v):
        nb = self.n_basis
        Hd = np.zeros((nb, nb))
        self.L.orc_brute_kinetic(ctypes.byref(self.sys), _d(np.ascontiguousarray(v, dtype=np.float64)), _d(Hd))
        return Hd

    # ---- O4
    def update_density(self, D_values, want_grad=False, batches=None):
        """(n[n_points], grad_n[3][n_points] or None); entries of batches not listed stay 0."""
        sel = self._sel(batches)
        D = np.ascontiguousarray(D_values, dtype=np.float64)
        n = np.zeros(self.n_points)
        gn = np.zeros((3, self.n_points)) if want_grad else None
        self.L.orc_update_density(ctypes.byref(self.sys), len(sel), _i(sel), _d(D), _d(n), _d(gn))
        return n, gn

    def density_hessian(self, D_values, batches=None):
        """hess_n[6][n_points] in the order (xx, yy, zz, xy, xz, yz); entries of batches not listed stay 0."""
        sel = self._sel(batches)
        D = np.ascontiguousarray(D_values, dtype=np.float64)
        H = np.zeros((6, self.n_points))
        self.L.orc_density_hessian(ctypes.byref(self.sys), len(sel), _i(sel), _d(D), _d(H))
        return H

    def partition_weights(self, xyz, owner, r_part):
        """w_owner(xyz) of the neighbour-restricted Stratmann partition (reading P5) over this system's atoms."""
        xyz = np.ascontiguousarray(xyz, dtype=np.float64)
        owner = np.ascontiguousarray(owner, dtype=np.int32)
        out = np.zeros(len(xyz))
        self.L.orc_partition_weights(ctypes.byref(self.sys), len(xyz), _d(xyz), _i(owner), float(r_part), _d(out))
        return out

    def bloch_fold(self, H_values, atom_home, atom_T, n_home, kpt):
        """Complex dense [n_hb][n_hb] matrix h_ij(k) = sum_IJ e^{ik.(T_J - T_I)} h^uc_IJ (Eq. 7, 11, 12)."""
        H = np.ascontiguousarray(H_values, dtype=np.float64)
        home = np.ascontiguousarray(atom_home, dtype=np.int32)
        T = np.ascontiguousarray(atom_T, dtype=np.float64)
        k = np.ascontiguousarray(kpt, dtype=np.float64)
        afp = np.zeros(self.sys.n_atoms + 1, dtype=np.int64)
        self.L.orc_atom_fn_ptr(ctypes.byref(self.sys), _l(afp))
        nhb = int(afp[n_home])
        re, im = np.zeros((nhb, nhb)), np.zeros((nhb, nhb))
        self.L.orc_bloch_fold(ctypes.byref(self.sys), _d(H), _i(home), _d(T), int(n_home), _d(k), _d(re), _d(im))
        return re + 1j * im

    # ---- brute force, tiny inputs
    def brute(self, v=None, g=None, D_dense=None, want_grad=False):
        """(H_dense or None, n or None, grad_n or None) with no batches, no culling, no block pattern."""
        nb = self.n_basis
        Hd = np.zeros((nb, nb)) if v is not None else None
        n = np.zeros(self.n_points) if D_dense is not None else None
        gn = np.zeros((3, self.n_points)) if (D_dense is not None and want_grad) else None
        v = None if v is None else np.ascontiguousarray(v, dtype=np.float64)
        g = None if g is None else np.ascontiguousarray(g, dtype=np.float64)
        Dd = None if D_dense is None else np.ascontiguousarray(D_dense, dtype=np.float64)
        self.L.orc_brute(ctypes.byref(self.sys), _d(v), _d(g), _d(Hd), _d(Dd), _d(n), _d(gn))
        return Hd, n, gn

    # ---- Pulay forces (Eq. 16, 18)
    def radial2(self, spline, d):
        R, dR, d2R = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        self.L.orc_radial2(ctypes.byref(self.sys), int(spline), float(d), ctypes.byref(R), ctypes.byref(dR), ctypes.byref(d2R))
        return R.value, dR.value, d2R.value

    def shell_hess_at_point(self, atom, shell, r):
        """(phi[2l+1], grad[2l+1][3], hess[2l+1][6] = xx, yy, zz, xy, xz, yz)"""
        l = int(self.keep["shell_l"][shell])
        r = np.ascontiguousarray(r, dtype=np.float64)
        phi, gr, he = np.zeros(2 * l + 1), np.zeros((2 * l + 1, 3)), np.zeros((2 * l + 1, 6))
        self.L.orc_shell_hess_at_point(ctypes.byref(self.sys), int(atom), int(shell), _d(r), _d(phi), _d(gr), _d(he))
        return phi, gr, he

    def pulay_forces(self, v, D_values, g=None, Q_values=None, batches=None, kinetic=False):
        """F[n_atoms][3] summed over the listed batches."""
        sel = self._sel(batches)
        v = np.ascontiguousarray(v, dtype=np.float64)
        g = None if g is None else np.ascontiguousarray(g, dtype=np.float64)
        D = np.ascontiguousarray(D_values, dtype=np.float64)
        Q = None if Q_values is None else np.ascontiguousarray(Q_values, dtype=np.float64)
        F = np.zeros((self.sys.n_atoms, 3))
        self.L.orc_pulay_forces(ctypes.byref(self.sys), len(sel), _i(sel), _d(v), _d(g), _d(D), _d(Q), int(bool(kinetic)), _d(F))
        return F

    def brute_forces(self, v, D_dense, g=None, Q_dense=None, kinetic=False):
        v = np.ascontiguousarray(v, dtype=np.float64)
        g = None if g is None else np.ascontiguousarray(g, dtype=np.float64)
        Dd = np.ascontiguousarray(D_dense, dtype=np.float64)
        Qd = None if Q_dense is None else np.ascontiguousarray(Q_dense, dtype=np.float64)
        F = np.zeros((self.sys.n_atoms, 3))
        self.L.orc_brute_forces(ctypes.byref(self.sys), _d(v), _d(g), _d(Dd), _d(Qd), int(bool(kinetic)), _d(F))
        return F

    def pulay_stress(self, v, D_values, g=None, Q_values=None, batches=None, kinetic=False, volume=1.0):
        """sigma[3][3] (O9): Pulay part of Eq. 20 summed over the listed batches; volume = 1 gives dE/d eps."""
        sel = self._sel(batches)
        v = np.ascontiguousarray(v, dtype=np.float64)
        g = None if g is None else np.ascontiguousarray(g, dtype=np.float64)
        D = np.ascontiguousarray(D_values, dtype=np.float64)
        Q = None if Q_values is None else np.ascontiguousarray(Q_values, dtype=np.float64)
        sig = np.zeros((3, 3))
        self.L.orc_pulay_stress(ctypes.byref(self.sys), len(sel), _i(sel), _d(v), _d(g), _d(D), _d(Q), int(bool(kinetic)),
                                float(volume), _d(sig))
        return sig

    def brute_stress(self, v, D_dense, g=None, Q_dense=None, volume=1.0, kinetic=False):
        v = np.ascontiguousarray(v, dtype=np.float64)
        g = None if g is None else np.ascontiguousarray(g, dtype=np.float64)
        Dd = np.ascontiguousarray(D_dense, dtype=np.float64)
        Qd = None if Q_dense is None else np.ascontiguousarray(Q_dense, dtype=np.float64)
        sig = np.zeros((3, 3))
        if kinetic:
            self.L.orc_brute_stress_ks(ctypes.byref(self.sys), _d(v), _d(g), _d(Dd), _d(Qd), 1, float(volume), _d(sig))
        else:
            self.L.orc_brute_stress(ctypes.byref(self.sys), _d(v), _d(g), _d(Dd), _d(Qd), float(volume), _d(sig))
        return sig
