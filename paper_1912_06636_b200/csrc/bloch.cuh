// bloch.cuh -- periodic boundary conditions: Bloch sums of the real-space matrix (Eq. 7,
// 11, 12 L85-113):   h_ij(k) = sum_{I image of i} sum_{J image of j} e^{ik.(T_J - T_I)} h^uc_IJ ,
// h^uc being the block-sparse matrix over the N_rs functions (cell atoms and their images) that
// aims_gpu_integrate_hamiltonian integrates unchanged.  One CTA per stored atom-pair block; a thread per element adds
// h e^{i theta} to (home_i, home_j) and -- the stored upper block also stands for its transpose -- h e^{-i theta} to
// (home_j, home_i).  Memory-bound and small (the value array is read once); FP64 atomics on the dense output.
#pragma once
#include "common.cuh"

namespace aims {

struct BlochBlock { long long off; int ld, nA, nB, i0, j0, diag; double cs, sn; };   // one stored block and its phase

__global__ void __launch_bounds__(128) k_bloch_fold(const BlochBlock *blocks, const double *H, int nhb, double *out_re,
                                                    double *out_im) {
  const BlochBlock B = blocks[blockIdx.x];
  for (int e = threadIdx.x; e < B.nA * B.nB; e += blockDim.x) {
    const int a = e / B.nB, b = e - a * B.nB;
    const double h = H[B.off + (long long)a * B.ld + b];
    const long long ij = (long long)(B.i0 + a) * nhb + (B.j0 + b);
    red_add_f64(out_re + ij, h * B.cs);
    red_add_f64(out_im + ij, h * B.sn);
    if (!B.diag) {
      const long long ji = (long long)(B.j0 + b) * nhb + (B.i0 + a);
      red_add_f64(out_re + ji, h * B.cs);
      red_add_f64(out_im + ji, -(h * B.sn));
    }
  }
}

}  // namespace aims
