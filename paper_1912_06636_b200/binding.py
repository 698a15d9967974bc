"""ctypes binding of libaims_gpu.so (include/aims_gpu.h).  Argument marshalling only: torch supplies device memory
and the stream; every step of the path runs in the library's CUDA kernels.  No CPU fallback, no other backend.
"""
from __future__ import annotations

import ctypes
import os
import re

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libaims_gpu.so")        # the product library; no environment variable changes this
HEADER_PATH = os.path.join(os.path.dirname(_HERE), "include", "aims_gpu.h")

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int32)
_lp = ctypes.POINTER(ctypes.c_int64)
_vp = ctypes.c_void_p


class AimsError(RuntimeError):
    pass


class _BasisDesc(ctypes.Structure):
    _fields_ = [("n_atoms", ctypes.c_int32), ("n_species", ctypes.c_int32), ("n_shells", ctypes.c_int32),
                ("n_splines", ctypes.c_int32), ("n_knots", ctypes.c_int32),
                ("atom_xyz", _dp), ("atom_species", _ip), ("species_shell_ptr", _ip), ("shell_l", _ip),
                ("shell_rcut", _dp), ("shell_spline", _ip), ("r0", ctypes.c_double), ("log_inc", ctypes.c_double),
                ("spline_coef", _dp)]


class _GridDesc(ctypes.Structure):
    _fields_ = [("n_points", ctypes.c_int64), ("n_batches", ctypes.c_int32), ("max_batch_points", ctypes.c_int32),
                ("xyz", _dp), ("w", _dp), ("batch_ptr", _lp)]


class _BsrDesc(ctypes.Structure):
    _fields_ = [("n_block_rows", ctypes.c_int32), ("row_ptr", _lp), ("col_atom", _ip), ("blk_off", _lp),
                ("blk_ld", _ip), ("n_values", ctypes.c_int64)]


_lib = None


def exported_symbols():
    """Names declared in include/aims_gpu.h (every `int|const char*|int64_t aims_gpu_*(`)."""
    with open(HEADER_PATH) as f:
        text = f.read()
    return sorted(set(re.findall(r"\b(aims_gpu_[a-z0-9_]+)\s*\(", text)))


def load_library(path=None, allow_probe=False):
    """dlopen libaims_gpu.so; raises (never falls back) if it is missing or lacks a declared symbol.
    path: another build of the same sources (build.py --define ... --tag ...), for the measurements under profiles/ only; it must
    be given before the first use of the binding.  A library that reports compile-time switches (aims_gpu_build_flags() != "")
    may compute something else than H and n on purpose and is refused unless allow_probe is set."""
    global _lib
    want = os.path.abspath(path) if path else LIB_PATH
    if _lib is not None:
        # one library per process: whoever loads first decides (bench.py --lib does it before anything else); a later call
        # without a path gets that library, a later call that names ANOTHER file is an error, never a silent swap
        if path and want != _lib._aims_path:
            raise AimsError("a different library is already loaded: %s" % _lib._aims_path)
        return _lib
    if not os.path.exists(want):
        raise AimsError("%s is not built: run `python -m paper_1912_06636_b200.build` "
                        "(nvcc, sm_100a). There is no CPU fallback." % os.path.basename(want))
    L = ctypes.CDLL(want)
    for name in exported_symbols():
        if not hasattr(L, name):
            raise AimsError("%s does not export %s" % (os.path.basename(want), name))
    L.aims_gpu_build_flags.restype = ctypes.c_char_p
    L.aims_gpu_build_flags.argtypes = []
    flags = L.aims_gpu_build_flags().decode()
    if flags and not allow_probe:
        raise AimsError("%s is a probe build (%s): its results are not the product's; pass allow_probe=True to measure with it"
                        % (want, flags))
    L._aims_path = want
    L._aims_build_flags = flags
    cp = _vp
    L.aims_gpu_create.restype = ctypes.c_int
    L.aims_gpu_create.argtypes = [ctypes.POINTER(cp), ctypes.POINTER(_BasisDesc), ctypes.POINTER(_GridDesc),
                                  ctypes.POINTER(_BsrDesc), ctypes.c_int, _vp, ctypes.c_int64]
    L.aims_gpu_destroy.restype = ctypes.c_int
    L.aims_gpu_destroy.argtypes = [cp]
    L.aims_gpu_last_error.restype = ctypes.c_char_p
    L.aims_gpu_last_error.argtypes = [cp]
    L.aims_gpu_basis_sizes.restype = ctypes.c_int
    L.aims_gpu_basis_sizes.argtypes = [cp, ctypes.c_int32, ctypes.c_int32, _lp, _lp]
    L.aims_gpu_eval_basis.restype = ctypes.c_int
    L.aims_gpu_eval_basis.argtypes = [cp, ctypes.c_int32, ctypes.c_int32, _vp, _vp, _vp, _vp, _vp]
    L.aims_gpu_integrate_hamiltonian.restype = ctypes.c_int
    L.aims_gpu_integrate_hamiltonian.argtypes = [cp, ctypes.c_int32, ctypes.c_int32, _vp, _vp, _vp, ctypes.c_int]
    L.aims_gpu_integrate_hamiltonian_ks.restype = ctypes.c_int
    L.aims_gpu_integrate_hamiltonian_ks.argtypes = [cp, ctypes.c_int32, ctypes.c_int32, _vp, _vp, ctypes.c_int, _vp, ctypes.c_int]
    L.aims_gpu_add_tau_matrix.restype = ctypes.c_int
    L.aims_gpu_add_tau_matrix.argtypes = [cp, ctypes.c_int32, ctypes.c_int32, _vp, _vp]
    L.aims_gpu_update_density.restype = ctypes.c_int
    L.aims_gpu_update_density.argtypes = [cp, ctypes.c_int32, ctypes.c_int32, _vp, _vp, _vp]
    L.aims_gpu_partition_weights.restype = ctypes.c_int
    L.aims_gpu_partition_weights.argtypes = [cp, ctypes.c_int64, _vp, _vp, ctypes.c_double, _vp]
    L.aims_gpu_partition_weights_noalloc.restype = ctypes.c_int
    L.aims_gpu_partition_weights_noalloc.argtypes = [ctypes.c_int, _vp, ctypes.c_int32, _vp, ctypes.c_int64, _vp, _vp, ctypes.c_double, _vp,
                                                     ctypes.c_char_p, ctypes.c_int32]
    L.aims_gpu_bloch_fold.restype = ctypes.c_int
    L.aims_gpu_bloch_fold.argtypes = [cp, _vp, _ip, _dp, ctypes.c_int32, _dp, _vp, _vp, ctypes.c_int]
    L.aims_gpu_density_hessian.restype = ctypes.c_int
    L.aims_gpu_density_hessian.argtypes = [cp, ctypes.c_int32, ctypes.c_int32, _vp, _vp]
    L.aims_gpu_pulay_forces.restype = ctypes.c_int
    L.aims_gpu_pulay_forces.argtypes = [cp, ctypes.c_int32, ctypes.c_int32, _vp, _vp, _vp, _vp, _vp, ctypes.c_int]
    L.aims_gpu_pulay_forces_ks.restype = ctypes.c_int
    L.aims_gpu_pulay_forces_ks.argtypes = [cp, ctypes.c_int32, ctypes.c_int32, _vp, _vp, ctypes.c_int, _vp, _vp, _vp, ctypes.c_int]
    L.aims_gpu_pulay_forces_stress.restype = ctypes.c_int
    L.aims_gpu_pulay_forces_stress.argtypes = [cp, ctypes.c_int32, ctypes.c_int32, _vp, _vp, ctypes.c_int, _vp, _vp,
                                               ctypes.c_double, _vp, _vp, ctypes.c_int]
    L.aims_gpu_synchronize.restype = ctypes.c_int
    L.aims_gpu_synchronize.argtypes = [cp]
    L.aims_gpu_batch_points.restype = ctypes.c_int
    L.aims_gpu_batch_points.argtypes = [ctypes.c_int, _vp, ctypes.c_int64, _vp, ctypes.c_int32, _vp, _lp, ctypes.c_int64, _ip]
    L.aims_gpu_periodic_images.restype = ctypes.c_int
    L.aims_gpu_periodic_images.argtypes = [_vp, ctypes.c_int32, _vp, ctypes.c_double, _vp, _vp, ctypes.c_int64, _lp]
    L.aims_gpu_wrap_points.restype = ctypes.c_int
    L.aims_gpu_wrap_points.argtypes = [ctypes.c_int, _vp, _vp, ctypes.c_int64, _vp]
    L.aims_gpu_set_deterministic.restype = ctypes.c_int
    L.aims_gpu_set_deterministic.argtypes = [cp, ctypes.c_int]
    L.aims_gpu_batch_nnz.restype = ctypes.c_int
    L.aims_gpu_batch_nnz.argtypes = [cp, _ip]
    L.aims_gpu_timing_enable.restype = ctypes.c_int
    L.aims_gpu_timing_enable.argtypes = [cp, ctypes.c_int]
    L.aims_gpu_timing_read.restype = ctypes.c_int
    L.aims_gpu_timing_read.argtypes = [cp, _dp, _lp]
    L.aims_gpu_stats.restype = ctypes.c_int
    L.aims_gpu_stats.argtypes = [cp, _lp, _ip, _ip, _dp, _dp, _dp]
    L.aims_gpu_launch_count.restype = ctypes.c_int64
    L.aims_gpu_launch_count.argtypes = [cp]
    L.aims_gpu_dmma_probe.restype = ctypes.c_int
    L.aims_gpu_dmma_probe.argtypes = [cp, ctypes.c_int, ctypes.c_int, _dp]
    L.aims_gpu_fp64_peak.restype = ctypes.c_int
    L.aims_gpu_fp64_peak.argtypes = [cp, ctypes.c_double, _dp]
    _lib = L
    return L


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


class Context:
    """One aims_gpu_ctx.  `bun` is any object with the attribute names of aims_synth.Bundle (numpy arrays)."""

    def __init__(self, bun, device=0, stream=None, workspace_bytes=0):
        import torch
        self.torch = torch
        self.L = load_library()
        if not torch.cuda.is_available():
            raise AimsError("no CUDA device: this path has no CPU fallback")
        self.device = torch.device("cuda", device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        f64 = lambda a: np.ascontiguousarray(a, dtype=np.float64)  # noqa: E731
        i32 = lambda a: np.ascontiguousarray(a, dtype=np.int32)    # noqa: E731
        i64 = lambda a: np.ascontiguousarray(a, dtype=np.int64)    # noqa: E731
        k = dict(atom_xyz=f64(bun.atom_xyz), atom_species=i32(bun.atom_species),
                 species_shell_ptr=i32(bun.species_shell_ptr), shell_l=i32(bun.shell_l), shell_rcut=f64(bun.shell_rcut),
                 shell_spline=i32(bun.shell_spline), spline_coef=f64(bun.spline_coef), xyz=f64(bun.xyz), w=f64(bun.w),
                 batch_ptr=i64(bun.batch_ptr), row_ptr=i64(bun.row_ptr), col_atom=i32(bun.col_atom),
                 blk_off=i64(bun.blk_off), blk_ld=i32(bun.blk_ld))
        d = lambda a: a.ctypes.data_as(_dp)   # noqa: E731
        i = lambda a: a.ctypes.data_as(_ip)   # noqa: E731
        l = lambda a: a.ctypes.data_as(_lp)   # noqa: E731
        self.n_points = int(k["xyz"].shape[0])
        self.n_batches = int(k["batch_ptr"].shape[0] - 1)
        self.n_values = int(bun.n_values)
        self.n_atoms = int(k["atom_xyz"].shape[0])
        self.batch_ptr = k["batch_ptr"]
        nfn_shell = 2 * k["shell_l"].astype(np.int64) + 1
        sp_nfn = np.array([nfn_shell[k["species_shell_ptr"][q]:k["species_shell_ptr"][q + 1]].sum()
                           for q in range(len(k["species_shell_ptr"]) - 1)], dtype=np.int64)
        self.atom_fn_ptr = np.concatenate([[0], np.cumsum(sp_nfn[k["atom_species"]])]).astype(np.int64)  # output sizes only
        bd = _BasisDesc(int(k["atom_xyz"].shape[0]), int(k["species_shell_ptr"].shape[0] - 1), int(k["shell_l"].shape[0]),
                        int(k["spline_coef"].shape[0]), int(bun.n_knots), d(k["atom_xyz"]), i(k["atom_species"]),
                        i(k["species_shell_ptr"]), i(k["shell_l"]), d(k["shell_rcut"]), i(k["shell_spline"]),
                        float(bun.r0), float(bun.log_inc), d(k["spline_coef"]))
        max_bp = int(np.diff(k["batch_ptr"]).max(initial=0))
        gd = _GridDesc(self.n_points, self.n_batches, max_bp, d(k["xyz"]), d(k["w"]), l(k["batch_ptr"]))
        pd = _BsrDesc(int(k["atom_xyz"].shape[0]), l(k["row_ptr"]), i(k["col_atom"]), l(k["blk_off"]), i(k["blk_ld"]),
                      self.n_values)
        self.h = ctypes.c_void_p()
        rc = self.L.aims_gpu_create(ctypes.byref(self.h), ctypes.byref(bd), ctypes.byref(gd), ctypes.byref(pd),
                                    int(device), ctypes.c_void_p(self.stream.cuda_stream), int(workspace_bytes))
        if rc != 0:
            msg = self.L.aims_gpu_last_error(self.h).decode() if self.h else ""
            if self.h:
                self.L.aims_gpu_destroy(self.h)
                self.h = None
            raise AimsError("aims_gpu_create failed (%d): %s" % (rc, msg))

    # ---- plumbing
    def _check(self, rc, what):
        if rc != 0:
            raise AimsError("%s failed (%d): %s" % (what, rc, self.L.aims_gpu_last_error(self.h).decode()))

    def _range(self, b0, b1):
        return int(b0), int(self.n_batches if b1 is None else b1)

    def close(self):
        if getattr(self, "h", None):
            self.L.aims_gpu_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def synchronize(self):
        self._check(self.L.aims_gpu_synchronize(self.h), "aims_gpu_synchronize")

    def set_deterministic(self, enable=True):
        self._check(self.L.aims_gpu_set_deterministic(self.h, int(bool(enable))), "aims_gpu_set_deterministic")

    def batch_nnz(self):
        out = np.zeros(max(self.n_batches, 1), dtype=np.int32)
        self._check(self.L.aims_gpu_batch_nnz(self.h, out.ctypes.data_as(_ip)), "aims_gpu_batch_nnz")
        return out[:self.n_batches]

    def timing_enable(self, enable=True):
        self._check(self.L.aims_gpu_timing_enable(self.h, int(bool(enable))), "aims_gpu_timing_enable")

    def timing_read(self):
        """{kernel: (device ms, launches)} since the last enable/read."""
        ms = (ctypes.c_double * 6)()
        ln = (ctypes.c_int64 * 6)()
        self._check(self.L.aims_gpu_timing_read(self.h, ms, ln), "aims_gpu_timing_read")
        names = ("k_cull", "k_eval", "k_hamiltonian", "k_density", "other", "k_forces")
        return {k: (ms[i], int(ln[i])) for i, k in enumerate(names)}

    def launch_count(self):
        return int(self.L.aims_gpu_launch_count(self.h))

    def stats(self):
        s, m, a = ctypes.c_int64(), ctypes.c_int32(), ctypes.c_int32()
        f1, f2, f3 = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        self._check(self.L.aims_gpu_stats(self.h, ctypes.byref(s), ctypes.byref(m), ctypes.byref(a), ctypes.byref(f1),
                                          ctypes.byref(f2), ctypes.byref(f3)), "aims_gpu_stats")
        return dict(sum_nnz=s.value, max_nnz=m.value, max_active_atoms=a.value, flops_h_lda=f1.value,
                    flops_h_gga=f2.value, flops_density=f3.value)

    def dmma_probe(self, variant, warps_per_sm):
        t = ctypes.c_double()
        self._check(self.L.aims_gpu_dmma_probe(self.h, int(variant), int(warps_per_sm), ctypes.byref(t)), "aims_gpu_dmma_probe")
        return t.value

    def fp64_peak(self, ms_target=200.0):
        t = ctypes.c_double()
        self._check(self.L.aims_gpu_fp64_peak(self.h, float(ms_target), ctypes.byref(t)), "aims_gpu_fp64_peak")
        return t.value

    def _dev(self, a, dtype=None):
        """Device copy of `a` on the CONTEXT stream (the stream the kernels run on): the copy is ordered before the
        kernels that read it, and the caching allocator ties the temporary to that stream."""
        torch = self.torch
        with torch.cuda.stream(self.stream):
            if isinstance(a, torch.Tensor):
                if a.device == self.device and a.is_contiguous() and (dtype is None or a.dtype == dtype):
                    return a
                t = a.to(self.device)
                return t.contiguous() if dtype is None else t.to(dtype).contiguous()
            return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).to(self.device)

    # ---- the three hot calls (device tensors in, device tensors out)
    def basis_sizes(self, b0=0, b1=None):
        b0, b1 = self._range(b0, b1)
        ni, nph = ctypes.c_int64(), ctypes.c_int64()
        self._check(self.L.aims_gpu_basis_sizes(self.h, b0, b1, ctypes.byref(ni), ctypes.byref(nph)), "aims_gpu_basis_sizes")
        return ni.value, nph.value

    def eval_basis(self, b0=0, b1=None, want_grad=False):
        """(fn_ptr, fn_index, phi_ptr, phi, dphi|None) as device tensors (layout: include/aims_gpu.h)."""
        torch = self.torch
        b0, b1 = self._range(b0, b1)
        ni, nph = self.basis_sizes(b0, b1)
        with torch.cuda.stream(self.stream):
            fn_ptr = torch.empty(b1 - b0 + 1, dtype=torch.int64, device=self.device)
            phi_ptr = torch.empty(b1 - b0 + 1, dtype=torch.int64, device=self.device)
            fn_index = torch.empty(max(ni, 1), dtype=torch.int32, device=self.device)
            phi = torch.empty(max(nph, 1), dtype=torch.float64, device=self.device)
            dphi = torch.empty(max(3 * nph, 1), dtype=torch.float64, device=self.device) if want_grad else None
        self._check(self.L.aims_gpu_eval_basis(self.h, b0, b1, _ptr(fn_ptr), _ptr(fn_index), _ptr(phi_ptr), _ptr(phi),
                                               _ptr(dphi)), "aims_gpu_eval_basis")
        return fn_ptr, fn_index[:ni], phi_ptr, phi[:nph], (dphi[:3 * nph] if want_grad else None)

    def integrate_hamiltonian(self, v, g=None, H=None, b0=0, b1=None, accumulate=False, kinetic=False):
        torch = self.torch
        b0, b1 = self._range(b0, b1)
        v = self._dev(v, torch.float64)
        g = None if g is None else self._dev(g, torch.float64)
        if v.numel() != self.n_points or (g is not None and g.numel() != 3 * self.n_points):
            raise AimsError("v must have n_points entries and g 3*n_points")
        if H is None:
            with torch.cuda.stream(self.stream):
                H = torch.empty(self.n_values, dtype=torch.float64, device=self.device)
            accumulate = False
        if kinetic:
            self._check(self.L.aims_gpu_integrate_hamiltonian_ks(self.h, b0, b1, _ptr(v), _ptr(g), 1, _ptr(H),
                                                                 int(bool(accumulate))), "aims_gpu_integrate_hamiltonian_ks")
            return H
        self._check(self.L.aims_gpu_integrate_hamiltonian(self.h, b0, b1, _ptr(v), _ptr(g), _ptr(H), int(bool(accumulate))),
                    "aims_gpu_integrate_hamiltonian")
        return H

    def add_tau_matrix(self, xi, H=None, b0=0, b1=None):
        """H += 1/2 sum_p w xi grad phi_i . grad phi_j (include/aims_gpu.h: aims_gpu_add_tau_matrix); H = None starts from zero."""
        torch = self.torch
        b0, b1 = self._range(b0, b1)
        xi = self._dev(xi, torch.float64)
        if xi.numel() != self.n_points:
            raise AimsError("xi must have n_points entries")
        if H is None:
            with torch.cuda.stream(self.stream):
                H = torch.zeros(self.n_values, dtype=torch.float64, device=self.device)
        self._check(self.L.aims_gpu_add_tau_matrix(self.h, b0, b1, _ptr(xi), _ptr(H)), "aims_gpu_add_tau_matrix")
        return H

    def update_density(self, D, want_grad=False, n=None, grad_n=None, b0=0, b1=None):
        torch = self.torch
        b0, b1 = self._range(b0, b1)
        D = self._dev(D, torch.float64)
        if D.numel() != self.n_values:
            raise AimsError("D must have n_values entries")
        with torch.cuda.stream(self.stream):
            if n is None:
                n = torch.zeros(self.n_points, dtype=torch.float64, device=self.device)
            if want_grad and grad_n is None:
                grad_n = torch.zeros((3, self.n_points), dtype=torch.float64, device=self.device)
        self._check(self.L.aims_gpu_update_density(self.h, b0, b1, _ptr(D), _ptr(n), _ptr(grad_n) if want_grad else None),
                    "aims_gpu_update_density")
        return n, (grad_n if want_grad else None)

    def partition_weights(self, xyz, owner, r_part):
        """w_owner(xyz) of the Stratmann partition over the context's atoms (include/aims_gpu.h: aims_gpu_partition_weights)."""
        torch = self.torch
        xyz = self._dev(xyz, torch.float64).reshape(-1, 3).contiguous()
        owner = self._dev(owner, torch.int32)
        if owner.numel() != xyz.shape[0]:
            raise AimsError("owner must have one entry per point")
        with torch.cuda.stream(self.stream):
            out = torch.empty(xyz.shape[0], dtype=torch.float64, device=self.device)
        self._check(self.L.aims_gpu_partition_weights(self.h, int(xyz.shape[0]), _ptr(xyz), _ptr(owner), float(r_part), _ptr(out)),
                    "aims_gpu_partition_weights")
        return out

    def bloch_fold(self, H, atom_home, atom_T, n_home, kpt, n_home_basis=None):
        """Complex device tensor [n_hb][n_hb]: Bloch sums of a real-space matrix (include/aims_gpu.h: aims_gpu_bloch_fold).
        n_hb = functions of the first n_home atoms (what the library writes); n_home_basis, if given, must agree."""
        torch = self.torch
        n_hb = int(self.atom_fn_ptr[int(n_home)])
        if n_home_basis is not None and int(n_home_basis) != n_hb:
            raise AimsError("n_home_basis %d != functions of the %d cell atoms (%d)" % (n_home_basis, n_home, n_hb))
        n_home_basis = n_hb
        H = self._dev(H, torch.float64)
        if H.numel() != self.n_values:
            raise AimsError("H must have n_values entries")
        home = np.ascontiguousarray(atom_home, dtype=np.int32)
        T = np.ascontiguousarray(atom_T, dtype=np.float64)
        k = np.ascontiguousarray(kpt, dtype=np.float64)
        if home.shape[0] != self.n_atoms or T.shape != (self.n_atoms, 3) or k.shape != (3,):
            raise AimsError("atom_home [n_atoms], atom_T [n_atoms][3], kpt [3]")
        with torch.cuda.stream(self.stream):
            re = torch.empty((n_home_basis, n_home_basis), dtype=torch.float64, device=self.device)
            im = torch.empty_like(re)
        self._check(self.L.aims_gpu_bloch_fold(self.h, _ptr(H), home.ctypes.data_as(_ip), T.ctypes.data_as(_dp), int(n_home),
                                               k.ctypes.data_as(_dp), _ptr(re), _ptr(im), 0), "aims_gpu_bloch_fold")
        return torch.complex(re, im)

    def density_hessian(self, D, hess_n=None, b0=0, b1=None):
        """hess_n[6][n_points] (xx, yy, zz, xy, xz, yz), device tensor (include/aims_gpu.h: aims_gpu_density_hessian)."""
        torch = self.torch
        b0, b1 = self._range(b0, b1)
        D = self._dev(D, torch.float64)
        if D.numel() != self.n_values:
            raise AimsError("D must have n_values entries")
        if hess_n is None:
            with torch.cuda.stream(self.stream):
                hess_n = torch.zeros((6, self.n_points), dtype=torch.float64, device=self.device)
        self._check(self.L.aims_gpu_density_hessian(self.h, b0, b1, _ptr(D), _ptr(hess_n)), "aims_gpu_density_hessian")
        return hess_n

    def pulay_forces(self, v, D, g=None, Q=None, F=None, b0=0, b1=None, accumulate=False, kinetic=False):
        """F[n_atoms][3] (device tensor): Pulay forces of batches [b0,b1) (include/aims_gpu.h: aims_gpu_pulay_forces)."""
        torch = self.torch
        b0, b1 = self._range(b0, b1)
        v = self._dev(v, torch.float64)
        D = self._dev(D, torch.float64)
        g = None if g is None else self._dev(g, torch.float64)
        Q = None if Q is None else self._dev(Q, torch.float64)
        if v.numel() != self.n_points or (g is not None and g.numel() != 3 * self.n_points):
            raise AimsError("v must have n_points entries and g 3*n_points")
        if D.numel() != self.n_values or (Q is not None and Q.numel() != self.n_values):
            raise AimsError("D and Q must have n_values entries")
        if F is None:
            with torch.cuda.stream(self.stream):
                F = torch.empty((self.n_atoms, 3), dtype=torch.float64, device=self.device)
            accumulate = False
        if kinetic:
            self._check(self.L.aims_gpu_pulay_forces_ks(self.h, b0, b1, _ptr(v), _ptr(g), 1, _ptr(D), _ptr(Q), _ptr(F),
                                                        int(bool(accumulate))), "aims_gpu_pulay_forces_ks")
            return F
        self._check(self.L.aims_gpu_pulay_forces(self.h, b0, b1, _ptr(v), _ptr(g), _ptr(D), _ptr(Q), _ptr(F),
                                                 int(bool(accumulate))), "aims_gpu_pulay_forces")
        return F

    def pulay_forces_stress(self, v, D, g=None, Q=None, volume=1.0, F=None, sigma=None, b0=0, b1=None, accumulate=False,
                            kinetic=False, want_forces=True):
        """(F[n_atoms][3] | None, sigma[3][3]) device tensors (include/aims_gpu.h: aims_gpu_pulay_forces_stress)."""
        torch = self.torch
        b0, b1 = self._range(b0, b1)
        v = self._dev(v, torch.float64)
        D = self._dev(D, torch.float64)
        g = None if g is None else self._dev(g, torch.float64)
        Q = None if Q is None else self._dev(Q, torch.float64)
        if v.numel() != self.n_points or (g is not None and g.numel() != 3 * self.n_points):
            raise AimsError("v must have n_points entries and g 3*n_points")
        if D.numel() != self.n_values or (Q is not None and Q.numel() != self.n_values):
            raise AimsError("D and Q must have n_values entries")
        with torch.cuda.stream(self.stream):
            if sigma is None:
                sigma = torch.zeros((3, 3), dtype=torch.float64, device=self.device)
                fresh = True
            else:
                fresh = False
            if F is None and want_forces:
                F = torch.zeros((self.n_atoms, 3), dtype=torch.float64, device=self.device)
            elif fresh and not accumulate and F is not None:
                pass
        self._check(self.L.aims_gpu_pulay_forces_stress(self.h, b0, b1, _ptr(v), _ptr(g), int(bool(kinetic)), _ptr(D), _ptr(Q),
                                                        float(volume), _ptr(F), _ptr(sigma), int(bool(accumulate))),
                    "aims_gpu_pulay_forces_stress")
        return F, sigma

    # ---- end-to-end with HOST buffers (pinned): H2D of v, g, D; the two calls; D2H of H, n, grad n
    def make_host_buffers(self, want_grad):
        torch = self.torch
        pin = dict(pin_memory=True, dtype=torch.float64)
        hb = dict(v=torch.empty(self.n_points, **pin), D=torch.empty(self.n_values, **pin),
                  H=torch.empty(self.n_values, **pin), n=torch.empty(self.n_points, **pin))
        if want_grad:
            hb["g"] = torch.empty((3, self.n_points), **pin)
            hb["grad_n"] = torch.empty((3, self.n_points), **pin)
        dv = {k: torch.empty_like(t, device=self.device) for k, t in hb.items()}
        return hb, dv

    def step_host(self, hb, dv, want_grad):
        """One pass of the whole hot path from pinned host inputs to pinned host outputs, on the context stream."""
        torch = self.torch
        with torch.cuda.stream(self.stream):
            dv["v"].copy_(hb["v"], non_blocking=True)
            dv["D"].copy_(hb["D"], non_blocking=True)
            if want_grad:
                dv["g"].copy_(hb["g"], non_blocking=True)
            self.integrate_hamiltonian(dv["v"], dv["g"] if want_grad else None, H=dv["H"], accumulate=False)
            self.update_density(dv["D"], want_grad=want_grad, n=dv["n"], grad_n=dv.get("grad_n"))
            hb["H"].copy_(dv["H"], non_blocking=True)
            hb["n"].copy_(dv["n"], non_blocking=True)
            if want_grad:
                hb["grad_n"].copy_(dv["grad_n"], non_blocking=True)


def aims_gpu_batch_points(xyz, max_batch_points, device=0, stream=None):
    """(order, batch_ptr): device int64 tensor [n] (position in the batched grid -> original point index) and a numpy
    int64 array [n_batches + 1] (include/aims_gpu.h: aims_gpu_batch_points).  xyz: [n][3] array or tensor."""
    import torch
    L = load_library()
    if not torch.cuda.is_available():
        raise AimsError("no CUDA device: this path has no CPU fallback")
    dev = torch.device("cuda", device)
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    with torch.cuda.stream(st):
        x = xyz if isinstance(xyz, torch.Tensor) else torch.as_tensor(np.ascontiguousarray(xyz, dtype=np.float64))
        x = x.to(dev, torch.float64).reshape(-1, 3).contiguous()
        n = int(x.shape[0])
        order = torch.empty(max(n, 1), dtype=torch.int64, device=dev)
    cap = 2 * ((n + int(max_batch_points) - 1) // max(int(max_batch_points), 1)) + 2
    ptr = np.zeros(cap, dtype=np.int64)
    nb = ctypes.c_int32()
    rc = L.aims_gpu_batch_points(int(device), ctypes.c_void_p(st.cuda_stream), n, _ptr(x), int(max_batch_points), _ptr(order),
                                 ptr.ctypes.data_as(_lp), cap, ctypes.byref(nb))
    if rc != 0:
        raise AimsError("aims_gpu_batch_points failed (%d)" % rc)
    return order[:n], ptr[: nb.value + 1].copy()


def aims_gpu_periodic_images(lattice, frac, reach):
    """(atom_home int32 [n], atom_n int32 [n][3]) of include/aims_gpu.h: aims_gpu_periodic_images (host arrays in, host arrays out)."""
    L = load_library()
    lat = np.ascontiguousarray(lattice, dtype=np.float64).reshape(3, 3)
    fr = np.ascontiguousarray(frac, dtype=np.float64).reshape(-1, 3)
    n = ctypes.c_int64()
    rc = L.aims_gpu_periodic_images(lat.ctypes.data_as(_vp), len(fr), fr.ctypes.data_as(_vp), float(reach), None, None, 0, ctypes.byref(n))
    if rc != 0:
        raise AimsError("aims_gpu_periodic_images failed (%d)" % rc)
    home = np.zeros(max(n.value, 1), dtype=np.int32)
    nn = np.zeros((max(n.value, 1), 3), dtype=np.int32)
    rc = L.aims_gpu_periodic_images(lat.ctypes.data_as(_vp), len(fr), fr.ctypes.data_as(_vp), float(reach), home.ctypes.data_as(_vp),
                                    nn.ctypes.data_as(_vp), n.value, ctypes.byref(n))
    if rc != 0:
        raise AimsError("aims_gpu_periodic_images failed (%d)" % rc)
    return home[: n.value], nn[: n.value]


def aims_gpu_wrap_points(lattice, xyz, device=0, stream=None):
    """Device tensor [n][3] of the points mapped into the cell at T = 0 (include/aims_gpu.h: aims_gpu_wrap_points).  A tensor
    argument on the device is wrapped in place and returned."""
    import torch
    L = load_library()
    if not torch.cuda.is_available():
        raise AimsError("no CUDA device: this path has no CPU fallback")
    dev = torch.device("cuda", device)
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    lat = np.ascontiguousarray(lattice, dtype=np.float64).reshape(3, 3)
    with torch.cuda.stream(st):
        x = xyz if isinstance(xyz, torch.Tensor) else torch.as_tensor(np.ascontiguousarray(xyz, dtype=np.float64))
        x = x.to(dev, torch.float64).reshape(-1, 3).contiguous()
    rc = L.aims_gpu_wrap_points(int(device), ctypes.c_void_p(st.cuda_stream), lat.ctypes.data_as(_vp), int(x.shape[0]), _ptr(x))
    if rc != 0:
        raise AimsError("aims_gpu_wrap_points failed (%d)" % rc)
    return x


def aims_gpu_partition_weights_noalloc(atom_xyz, xyz, owner, r_part, w_part=None, device=0, stream=None):
    """Device tensor [n] of partition-of-unity weights, computed without the library allocating any device memory
    (include/aims_gpu.h: aims_gpu_partition_weights_noalloc).  For programs that cannot let a library call cudaMalloc: a rank
    at its MPS memory limit, a host whose pool allocator already owns the HBM, a loop that must not stall in the allocator.
    No context is needed; atom_xyz is a HOST array [n_atoms][3].  Pass xyz, owner and w_part as device tensors (float64
    [n][3], int32 [n], float64 [n]) and the call touches no allocator at all; host arrays are copied to the device through
    torch first and a missing w_part is made with torch, both for convenience only.  The library's built-in scratch array is
    shared by every call on the device: do not run two of these calls concurrently on one GPU.  Waits for the stream.
    Raises AimsError with the library's message when a size limit (AIMS_NOALLOC_MAX_ATOMS / _MAX_CELLS) is exceeded."""
    import torch
    L = load_library()
    if not torch.cuda.is_available():
        raise AimsError("no CUDA device: this path has no CPU fallback")
    dev = torch.device("cuda", device)
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    R = np.ascontiguousarray(atom_xyz, dtype=np.float64).reshape(-1, 3)
    with torch.cuda.stream(st):
        x = xyz if isinstance(xyz, torch.Tensor) else torch.as_tensor(np.ascontiguousarray(xyz, dtype=np.float64))
        x = x.to(dev, torch.float64).reshape(-1, 3).contiguous()
        o = owner if isinstance(owner, torch.Tensor) else torch.as_tensor(np.ascontiguousarray(owner, dtype=np.int32))
        o = o.to(dev, torch.int32).contiguous()
        n = int(x.shape[0])
        if o.numel() != n:
            raise AimsError("owner must have one entry per point")
        if w_part is None:
            w_part = torch.empty(n, dtype=torch.float64, device=dev)
    if w_part.dtype != torch.float64 or w_part.device != dev or w_part.numel() != n or not w_part.is_contiguous():
        raise AimsError("w_part must be a contiguous float64 tensor of n entries on the device")
    msg = ctypes.create_string_buffer(512)
    rc = L.aims_gpu_partition_weights_noalloc(int(device), ctypes.c_void_p(st.cuda_stream), int(R.shape[0]), R.ctypes.data_as(_vp), n,
                                              _ptr(x) if n else None, _ptr(o) if n else None, float(r_part), _ptr(w_part) if n else None,
                                              msg, len(msg))
    if rc != 0:
        raise AimsError("aims_gpu_partition_weights_noalloc failed (%d): %s" % (rc, msg.value.decode(errors="replace")))
    return w_part


# ---- module-level functions with the names of the C ABI
def aims_gpu_create(bun, device=0, stream=None, workspace_bytes=0):
    return Context(bun, device, stream, workspace_bytes)


def aims_gpu_destroy(ctx):
    ctx.close()


def aims_gpu_eval_basis(ctx, b0=0, b1=None, want_grad=False):
    return ctx.eval_basis(b0, b1, want_grad)


def aims_gpu_integrate_hamiltonian(ctx, v, g=None, H=None, b0=0, b1=None, accumulate=False):
    return ctx.integrate_hamiltonian(v, g, H, b0, b1, accumulate)


def aims_gpu_integrate_hamiltonian_ks(ctx, v, g=None, kinetic=True, H=None, b0=0, b1=None, accumulate=False):
    return ctx.integrate_hamiltonian(v, g, H, b0, b1, accumulate, kinetic=kinetic)


def aims_gpu_add_tau_matrix(ctx, xi, H=None, b0=0, b1=None):
    return ctx.add_tau_matrix(xi, H, b0, b1)


def aims_gpu_update_density(ctx, D, want_grad=False, n=None, grad_n=None, b0=0, b1=None):
    return ctx.update_density(D, want_grad, n, grad_n, b0, b1)


def aims_gpu_partition_weights(ctx, xyz, owner, r_part):
    return ctx.partition_weights(xyz, owner, r_part)


def aims_gpu_set_deterministic(ctx, enable=True):
    ctx.set_deterministic(enable)


def aims_gpu_bloch_fold(ctx, H, atom_home, atom_T, n_home, kpt, n_home_basis=None):
    return ctx.bloch_fold(H, atom_home, atom_T, n_home, kpt, n_home_basis)


def aims_gpu_density_hessian(ctx, D, hess_n=None, b0=0, b1=None):
    return ctx.density_hessian(D, hess_n, b0, b1)


def aims_gpu_pulay_forces(ctx, v, D, g=None, Q=None, F=None, b0=0, b1=None, accumulate=False):
    return ctx.pulay_forces(v, D, g, Q, F, b0, b1, accumulate)


def aims_gpu_pulay_forces_stress(ctx, v, D, g=None, kinetic=False, Q=None, volume=1.0, F=None, sigma=None, b0=0, b1=None,
                                 accumulate=False):
    return ctx.pulay_forces_stress(v, D, g, Q, volume, F, sigma, b0, b1, accumulate, kinetic)


def aims_gpu_pulay_forces_ks(ctx, v, D, g=None, kinetic=True, Q=None, F=None, b0=0, b1=None, accumulate=False):
    return ctx.pulay_forces(v, D, g, Q, F, b0, b1, accumulate, kinetic=kinetic)
