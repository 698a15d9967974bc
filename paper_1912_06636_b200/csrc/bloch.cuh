// bloch.cuh -- periodic boundary conditions: Bloch sums of the real-space matrix (Eq. 7,
// 11, 12 L85-113):   h_ij(k) = sum_{I image of i} sum_{J image of j} e^{ik.(T_J - T_I)} h^uc_IJ ,
// h^uc being the block-sparse matrix over the N_rs functions (cell atoms and their images) that
// aims_gpu_integrate_hamiltonian integrates unchanged.
// Output-stationary: one CTA per pair (cell atom hi, cell atom hj) walks the list of stored blocks (A, B) with
// home(A) = hi, home(B) = hj -- and, the stored upper block also standing for its transpose, the blocks (B, A) with
// home(B) = hi, home(A) = hj read transposed with the conjugate phase -- in a fixed order, a thread per matrix element, and
// writes its tile once.  No atomics (round 1 added 4 REDs per stored value to the dense output: 65 ms per k-point on the
// 54-atom supercell, now < 1 ms), bitwise reproducible.  The lists depend on atom_home only and are cached in the context.
#pragma once
#include "common.cuh"

namespace aims {

struct BlochContrib { long long off; int ld, A, B, transposed; };   // stored block (A, B >= A) feeding one (hi, hj) tile

__global__ void __launch_bounds__(128) k_bloch_fold(const BlochContrib *contrib, const int *tile_ptr, const int *atom_fn_ptr,
                                                    const double *atom_T, double kx, double ky, double kz, const double *H,
                                                    int n_home, int nhb, double *out_re, double *out_im, int accumulate) {
  const int hi = blockIdx.x / n_home, hj = blockIdx.x - hi * n_home;
  const int i0 = atom_fn_ptr[hi], nA = atom_fn_ptr[hi + 1] - i0, j0 = atom_fn_ptr[hj], nB = atom_fn_ptr[hj + 1] - j0;
  const int c0 = tile_ptr[blockIdx.x], c1 = tile_ptr[blockIdx.x + 1];
  for (int e = threadIdx.x; e < nA * nB; e += blockDim.x) {
    const int a = e / nB, b = e - a * nB;
    double re = 0.0, im = 0.0;
    for (int c = c0; c < c1; c++) {
      const BlochContrib C = contrib[c];
      const double th = kx * (atom_T[3 * C.B] - atom_T[3 * C.A]) + ky * (atom_T[3 * C.B + 1] - atom_T[3 * C.A + 1]) +
                        kz * (atom_T[3 * C.B + 2] - atom_T[3 * C.A + 2]);
      double sn, cs;
      sincos(th, &sn, &cs);
      // direct: tile element (a, b) = block[a][b], phase e^{+i theta}; transposed: tile element (a, b) = block[b][a], e^{-i theta}
      const double h = C.transposed ? H[C.off + (long long)b * C.ld + a] : H[C.off + (long long)a * C.ld + b];
      re += h * cs;
      im += C.transposed ? -(h * sn) : h * sn;
    }
    const long long ij = (long long)(i0 + a) * nhb + (j0 + b);
    if (accumulate) { out_re[ij] += re; out_im[ij] += im; }
    else { out_re[ij] = re; out_im[ij] = im; }
  }
}

}  // namespace aims
