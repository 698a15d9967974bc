"""Paper-style CPU path: what the CPU column of Fig. 6 does -- per batch, evaluate phi on
nnz(B), then ONE dense BLAS call per product:
    integration   w -> K = diag(w) phi (L325 "dgmm"), h_batch = DSYR2K(h_times_phi, K) (L326), insert_into_h (L327)
    density       density_mat = D restricted to nnz(B) (L357), temp = DSYMM(density_mat, phi) (L359), n = sum_i temp*phi (L360)
through numpy's BLAS (matmul -> dgemm on the host's cores).

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rule as oracle/aims_oracle.c): a second, reported CPU baseline for bench.py
 and an independent cross-check of the triple-loop oracle (tests/test_oracle_blas_crosscheck.py,
<= 1e-12).  phi, grad phi and nnz(B) come from the oracle's own O1/O2 routines; the contractions here are library calls.
It imports nothing from paper_1912_06636_b200.
"""
import numpy as np

from .oracle import Oracle


class BlasBaseline:
    def __init__(self, bun):
        self.bun = bun
        self.orc = Oracle(bun)
        self.nb = int(self.orc.n_basis)

    def dense(self, values):
        """Full symmetric matrix of a block-sparse value array (set-up, outside any timed region)."""
        from aims_synth import bsr_to_dense
        return bsr_to_dense(self.bun, values)

    def hamiltonian_dense(self, v, g=None, batches=None, out=None):
        """Dense H (n_basis x n_basis) summed over the listed batches: Eq. 23-27 with one matmul pair per batch."""
        bun, orc = self.bun, self.orc
        H = np.zeros((self.nb, self.nb)) if out is None else out
        for b in (range(bun.n_batches) if batches is None else batches):
            b = int(b)
            idx, phi, dphi = orc.eval_basis(b, want_grad=g is not None)
            if len(idx) == 0 or phi.shape[1] == 0:
                continue
            p0, p1 = int(bun.batch_ptr[b]), int(bun.batch_ptr[b + 1])
            w = bun.w[p0:p1]
            K = phi * w                                              # "dgmm": K_ir = w(r) phi_i(r), Eq. 25
            if g is None:
                L = phi * v[p0:p1]                                   # h phi = v phi
                hb = K @ L.T                                         # symmetric: DSYRK-shaped
            else:
                # L = 1/2 v phi + g.grad phi ; h_b = K L^T + L K^T   (DSYR2K, Fig. 6a)
                L = 0.5 * v[p0:p1] * phi + np.einsum("cp,cip->ip", g[:, p0:p1], dphi)
                M = K @ L.T
                hb = M + M.T
            H[np.ix_(idx, idx)] += hb                                # "insert_into_h"
        return H

    def density(self, D_dense, want_grad=False, batches=None):
        """n [n_points] (and grad n [3][n_points]) on the listed batches: DSYMM + row dots (Fig. 6b)."""
        bun, orc = self.bun, self.orc
        n = np.zeros(bun.n_points)
        gn = np.zeros((3, bun.n_points)) if want_grad else None
        for b in (range(bun.n_batches) if batches is None else batches):
            b = int(b)
            idx, phi, dphi = orc.eval_basis(b, want_grad=want_grad)
            if len(idx) == 0 or phi.shape[1] == 0:
                continue
            p0, p1 = int(bun.batch_ptr[b]), int(bun.batch_ptr[b + 1])
            Db = D_dense[np.ix_(idx, idx)]                           # "calculate_density_mat"
            T = Db @ phi                                             # DSYMM
            n[p0:p1] = (T * phi).sum(axis=0)
            if want_grad:
                gn[:, p0:p1] = 2.0 * np.einsum("cip,ip->cp", dphi, T)
        return n, gn
