// partition.cuh -- partition of unity of the atom-centred integration grids (Eq. 21-22
// L192-200; reading P5: Stratmann-Scuseria-Frisch cell function, a = 0.64, restricted to the atoms within r_part
// of the point).  The paper evaluates w(r) on the CPU before the batch loops; here one thread per point:
//   1. scan the atoms: nearest candidate and candidate count;
//   2. for every candidate A: P_A = prod_{B candidate, B != A} s(mu_AB), nearest atom first -- it zeroes most far atoms at
//      once, and the inner scan is skipped as soon as the product is exactly 0;
//   3. w_owner = P_owner / sum_A P_A.
// Atom coordinates are read through the read-only path (a few thousand doubles: L1-resident).  ALU / latency bound and far
// from the hot path (config 5: ~8 M points x ~60 candidates).
#pragma once
#include "common.cuh"

namespace aims {

__device__ __forceinline__ double stratmann_s(double mu) {
  const double x = mu / 0.64;
  if (x <= -1.0) return 1.0;
  if (x >= 1.0) return 0.0;
  const double x2 = x * x;
  const double z = x * (35.0 + x2 * (-35.0 + x2 * (21.0 - 5.0 * x2))) / 16.0;
  return fmin(fmax(0.5 * (1.0 - z), 0.0), 1.0);
}

__global__ void __launch_bounds__(256) k_partition_weights(int n_atoms, const double *__restrict__ atom_xyz, long long n,
                                                           const double *__restrict__ xyz, const int *__restrict__ owner,
                                                           double r_part, double *__restrict__ out) {
  const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const double x = xyz[3 * p], y = xyz[3 * p + 1], z = xyz[3 * p + 2];
  auto dist = [&](int a, double &ax, double &ay, double &az) {
    ax = __ldg(atom_xyz + 3 * a); ay = __ldg(atom_xyz + 3 * a + 1); az = __ldg(atom_xyz + 3 * a + 2);
    // separately rounded operations in a fixed order: membership in cand(r) (d <= r_part) is a discrete decision
    const double dx = x - ax, dy = y - ay, dz = z - az;
    return sqrt(__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)));
  };
  int near = -1;
  double dnear = 1e300, nx = 0.0, ny = 0.0, nz = 0.0;
  for (int a = 0; a < n_atoms; a++) {
    double ax, ay, az;
    const double d = dist(a, ax, ay, az);
    if (d <= r_part && d < dnear) { dnear = d; near = a; nx = ax; ny = ay; nz = az; }
  }
  const int own = owner[p];
  double sum = 0.0, pown = 0.0;
  if (near >= 0) {
    for (int a = 0; a < n_atoms; a++) {
      double ax, ay, az;
      const double da = dist(a, ax, ay, az);
      if (da > r_part) continue;
      double P = 1.0;
      if (a != near) P = stratmann_s((da - dnear) / sqrt((ax - nx) * (ax - nx) + (ay - ny) * (ay - ny) + (az - nz) * (az - nz)));
      for (int b = 0; b < n_atoms && P != 0.0; b++) {
        if (b == a || b == near) continue;
        double bx, by, bz;
        const double db = dist(b, bx, by, bz);
        if (db > r_part) continue;
        P *= stratmann_s((da - db) / sqrt((ax - bx) * (ax - bx) + (ay - by) * (ay - by) + (az - bz) * (az - bz)));
      }
      sum += P;
      if (a == own) pown = P;
    }
  }
  out[p] = sum > 0.0 ? pown / sum : 0.0;
}

}  // namespace aims
