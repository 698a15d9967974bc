// partition.cuh -- partition of unity of the atom-centred integration grids (Eq. 21-22
// L192-200; reading P5: Stratmann-Scuseria-Frisch cell function, a = 0.64, restricted to the atoms within r_part
// of the point).  The paper evaluates w(r) on the CPU before the batch loops and stresses that the restriction to nearby
// atoms makes it O(N) (L190, L200).  Here:
//   host   a cell list of the atoms with cell edge r_part (counting sort; a few thousand atoms at most);
//   k_partition_weights   ONE WARP PER POINT:
//     1. the 27 cells around the point's cell -> candidates with d <= r_part (warp ballot compaction into shared memory),
//        put into ascending atom order (rank sort) so that every product below runs in the order the definition states;
//     2. lane A computes P_A = prod_{B candidate, B != A} s(mu_AB): nearest atom first -- it zeroes most far atoms at
//        once -- and the scan stops at an exact zero;  3. w_owner = P_owner / sum_A P_A  (warp shuffle sum).
// Work per point O(n_cand^2 / 32) per lane, independent of the number of atoms.  Membership d <= r_part is decided in
// separately rounded operations in a fixed order (a discrete decision, like reading P6).
#pragma once
#include "common.cuh"

namespace aims {

constexpr int kPartMaxCand = 256;     // atoms within r_part of one point
constexpr int kPartWarps = 8;

struct PartCells {
  double ox, oy, oz, inv_edge;   // origin and 1 / cell edge (edge >= r_part)
  int nx, ny, nz;
  const int *cell_start;         // [nx*ny*nz + 1]
  const int *cell_atom;          // [n_atoms] atoms sorted by cell
};

__device__ __forceinline__ double stratmann_s(double mu) {
  const double x = mu / 0.64;
  if (x <= -1.0) return 1.0;
  if (x >= 1.0) return 0.0;
  const double x2 = x * x;
  const double z = x * (35.0 + x2 * (-35.0 + x2 * (21.0 - 5.0 * x2))) / 16.0;
  return fmin(fmax(0.5 * (1.0 - z), 0.0), 1.0);
}

__global__ void __launch_bounds__(kPartWarps * 32) k_partition_weights(PartCells C, const double *__restrict__ atom_xyz, long long n,
                                                                      const double *__restrict__ xyz, const int *__restrict__ owner,
                                                                      double r_part, double *__restrict__ out, int *error_flag) {
  __shared__ int s_atom[kPartWarps][kPartMaxCand], s_tmp[kPartWarps][kPartMaxCand];
  __shared__ double s_d[kPartWarps][kPartMaxCand], s_dt[kPartWarps][kPartMaxCand];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long p = (long long)blockIdx.x * kPartWarps + warp;
  if (p >= n) return;
  const double x = xyz[3 * p], y = xyz[3 * p + 1], z = xyz[3 * p + 2];
  int *cat = s_atom[warp], *tat = s_tmp[warp];
  double *cd = s_d[warp], *td = s_dt[warp];

  // 1. candidates from the 27 cells around the point (cells outside the atom box hold nothing)
  // cell of the point, clamped to two cells outside the atom box (farther out nothing is within r_part anyway)
  const int cx = (int)fmin(fmax(floor((x - C.ox) * C.inv_edge), -2.0), (double)C.nx + 1.0);
  const int cy = (int)fmin(fmax(floor((y - C.oy) * C.inv_edge), -2.0), (double)C.ny + 1.0);
  const int cz = (int)fmin(fmax(floor((z - C.oz) * C.inv_edge), -2.0), (double)C.nz + 1.0);
  int ncand = 0;
  for (int dz = -1; dz <= 1; dz++)
    for (int dy = -1; dy <= 1; dy++) {
      const int iy = cy + dy, iz = cz + dz;
      if (iy < 0 || iy >= C.ny || iz < 0 || iz >= C.nz) continue;
      // the three x-neighbours are consecutive cells: one contiguous run of atoms
      const int x0 = max(cx - 1, 0), x1 = min(cx + 1, C.nx - 1);
      if (x0 > x1) continue;
      const int c0 = (iz * C.ny + iy) * C.nx + x0, c1 = (iz * C.ny + iy) * C.nx + x1;
      const int a0 = C.cell_start[c0], a1 = C.cell_start[c1 + 1];
      for (int base = a0; base < a1; base += 32) {
        const int k = base + lane;
        int a = -1;
        double d = 0.0;
        if (k < a1) {
          a = C.cell_atom[k];
          const double ddx = x - __ldg(atom_xyz + 3 * a), ddy = y - __ldg(atom_xyz + 3 * a + 1), ddz = z - __ldg(atom_xyz + 3 * a + 2);
          d = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(ddx, ddx), __dmul_rn(ddy, ddy)), __dmul_rn(ddz, ddz)));
          if (!(d <= r_part)) a = -1;
        }
        const unsigned m = __ballot_sync(0xffffffffu, a >= 0);
        if (a >= 0) {
          const int pos = ncand + __popc(m & ((1u << lane) - 1u));
          if (pos < kPartMaxCand) { tat[pos] = a; td[pos] = d; }
        }
        ncand += __popc(m);
      }
    }
  if (ncand > kPartMaxCand) {
    if (lane == 0) { atomicExch(error_flag, 5); out[p] = 0.0; }
    return;
  }
  __syncwarp();
  // ascending atom order (rank sort; atom indices are distinct)
  for (int i = lane; i < ncand; i += 32) {
    const int a = tat[i];
    int rank = 0;
    for (int j = 0; j < ncand; j++) rank += tat[j] < a;
    cat[rank] = a; cd[rank] = td[i];
  }
  __syncwarp();
  if (ncand == 0) { if (lane == 0) out[p] = 0.0; return; }
  // nearest candidate (first of equal distances in ascending atom order, as a sequential scan finds it)
  int inear = 0;
  double dnear = cd[0];
  for (int j = 1; j < ncand; j++)
    if (cd[j] < dnear) { dnear = cd[j]; inear = j; }
  const int anear = cat[inear];
  const double nx = __ldg(atom_xyz + 3 * anear), ny = __ldg(atom_xyz + 3 * anear + 1), nz = __ldg(atom_xyz + 3 * anear + 2);

  // 2. P_A for candidate A = lane, lane + 32, ...
  const int own = owner[p];
  double sum = 0.0, pown = 0.0;
  for (int i = lane; i < ncand; i += 32) {
    const int a = cat[i];
    const double da = cd[i];
    const double ax = __ldg(atom_xyz + 3 * a), ay = __ldg(atom_xyz + 3 * a + 1), az = __ldg(atom_xyz + 3 * a + 2);
    double P = 1.0;
    if (i != inear) P = stratmann_s((da - dnear) / sqrt((ax - nx) * (ax - nx) + (ay - ny) * (ay - ny) + (az - nz) * (az - nz)));
    for (int j = 0; j < ncand && P != 0.0; j++) {
      if (j == i || j == inear) continue;
      const int b = cat[j];
      const double bx = __ldg(atom_xyz + 3 * b), by = __ldg(atom_xyz + 3 * b + 1), bz = __ldg(atom_xyz + 3 * b + 2);
      P *= stratmann_s((da - cd[j]) / sqrt((ax - bx) * (ax - bx) + (ay - by) * (ay - by) + (az - bz) * (az - bz)));
    }
    sum += P;
    if (a == own) pown = P;
  }
  // 3. normalise
  for (int o = 16; o > 0; o >>= 1) {
    sum += __shfl_xor_sync(0xffffffffu, sum, o);
    pown += __shfl_xor_sync(0xffffffffu, pown, o);
  }
  if (lane == 0) out[p] = sum > 0.0 ? pown / sum : 0.0;
}

}  // namespace aims
