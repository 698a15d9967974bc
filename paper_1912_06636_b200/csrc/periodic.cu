// periodic.cu -- the two geometric steps of the periodic real-space path (Eq. 11-12):
//   aims_gpu_periodic_images   which periodic images of the cell atoms carry functions "that are non-zero on the unit cell" (L109-113),
//   aims_gpu_wrap_points       "each integration point r is mapped back to its periodic image within the unit cell at T = (0,0,0)"
//                              (L113-115), on the device.
// The paper states neither rule; reading P23 fixes both (see include/aims_gpu.h).  Product code: shares nothing with oracle/.
#include "../../include/aims_gpu.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <new>
#include <vector>

#include <cuda_runtime.h>

namespace {

struct Inv3 { double a[9], inv[9]; };

// r -> r A^-1 -> fractional part -> back to Cartesian; every product and sum separately rounded, sums left to right
__global__ void __launch_bounds__(256) k_wrap_points(Inv3 M, long long n, double *__restrict__ xyz) {
  const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const double x = xyz[3 * p], y = xyz[3 * p + 1], z = xyz[3 * p + 2];
  double f[3];
#pragma unroll
  for (int j = 0; j < 3; j++) {
    const double t = __dadd_rn(__dadd_rn(__dmul_rn(x, M.inv[j]), __dmul_rn(y, M.inv[3 + j])), __dmul_rn(z, M.inv[6 + j]));
    const double d = __dsub_rn(t, floor(t));
    f[j] = d >= 1.0 ? 0.0 : d;              // t = -tiny: 1 - tiny rounds to 1.0, the excluded face; it is the f = 0 face of the next cell
  }
#pragma unroll
  for (int j = 0; j < 3; j++)
    xyz[3 * p + j] = __dadd_rn(__dadd_rn(__dmul_rn(f[0], M.a[j]), __dmul_rn(f[1], M.a[3 + j])), __dmul_rn(f[2], M.a[6 + j]));
}

// cofactors with cyclic indices (the sign is already right), determinant along the first row
bool invert3(const double *a, double *inv) {
  double cof[9];
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) {
      const int r0 = (i + 1) % 3, r1 = (i + 2) % 3, c0 = (j + 1) % 3, c1 = (j + 2) % 3;
      const volatile double p = a[3 * r0 + c0] * a[3 * r1 + c1], q = a[3 * r0 + c1] * a[3 * r1 + c0];   // volatile: no contraction
      cof[3 * i + j] = p - q;
    }
  const volatile double t0 = a[0] * cof[0], t1 = a[1] * cof[1], t2 = a[2] * cof[2];
  const volatile double s01 = t0 + t1;
  const double det = s01 + t2;
  if (!(std::fabs(det) > 0.0)) return false;
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) inv[3 * i + j] = cof[3 * j + i] / det;
  return true;
}

double norm3(const double *v) { return std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]); }
void cross3(const double *u, const double *v, double *w) {
  w[0] = u[1] * v[2] - u[2] * v[1]; w[1] = u[2] * v[0] - u[0] * v[2]; w[2] = u[0] * v[1] - u[1] * v[0];
}

}  // namespace

extern "C" {

int aims_gpu_periodic_images(const double *lattice, int32_t n_home, const double *frac, double reach, int32_t *atom_home,
                             int32_t *atom_n, int64_t capacity, int64_t *n_atoms) {
  if (!lattice || !frac || !n_atoms || n_home <= 0 || !(reach >= 0.0) || capacity < 0 || (capacity > 0 && (!atom_home || !atom_n)))
    return AIMS_ERR_INVALID_ARG;
  try {
    double c12[3], vol, h[3], delta[3];
    cross3(lattice + 3, lattice + 6, c12);
    vol = std::fabs(lattice[0] * c12[0] + lattice[1] * c12[1] + lattice[2] * c12[2]);
    if (!(vol > 0.0)) return AIMS_ERR_INVALID_ARG;
    // the search box below (nmax) is sized for cell atoms inside the cell: unwrapped coordinates would silently lose images
    for (int a = 0; a < n_home; a++)
      for (int i = 0; i < 3; i++)
        if (!(frac[3 * a + i] >= 0.0 && frac[3 * a + i] < 1.0)) return AIMS_ERR_INVALID_ARG;
    int nmax[3];
    for (int i = 0; i < 3; i++) {
      double w[3];
      cross3(lattice + 3 * ((i + 1) % 3), lattice + 3 * ((i + 2) % 3), w);
      h[i] = vol / norm3(w);
      delta[i] = reach / h[i];
      nmax[i] = (int)std::ceil(delta[i] + 1.0);
    }
    struct Img { int far, n1, n2, n3, a; };
    std::vector<Img> out;
    for (int n1 = -nmax[0]; n1 <= nmax[0]; n1++)
      for (int n2 = -nmax[1]; n2 <= nmax[1]; n2++)
        for (int n3 = -nmax[2]; n3 <= nmax[2]; n3++)
          for (int a = 0; a < n_home; a++) {
            const double ff[3] = {frac[3 * a] + n1, frac[3 * a + 1] + n2, frac[3 * a + 2] + n3};
            bool keep = true;
            for (int i = 0; i < 3; i++) keep = keep && ff[i] > -delta[i] && ff[i] < 1.0 + delta[i];
            if (keep) out.push_back(Img{(n1 || n2 || n3) ? 1 : 0, n1, n2, n3, a});
          }
    std::sort(out.begin(), out.end(), [](const Img &x, const Img &y) {
      if (x.far != y.far) return x.far < y.far;
      if (x.n1 != y.n1) return x.n1 < y.n1;
      if (x.n2 != y.n2) return x.n2 < y.n2;
      if (x.n3 != y.n3) return x.n3 < y.n3;
      return x.a < y.a;
    });
    *n_atoms = (int64_t)out.size();
    if ((int64_t)out.size() > capacity) return capacity == 0 ? AIMS_OK : AIMS_ERR_INVALID_ARG;   // capacity 0: size query
    for (size_t k = 0; k < out.size(); k++) {
      atom_home[k] = out[k].a;
      atom_n[3 * k] = out[k].n1; atom_n[3 * k + 1] = out[k].n2; atom_n[3 * k + 2] = out[k].n3;
    }
    return AIMS_OK;
  } catch (const std::bad_alloc &) {
    return AIMS_ERR_NOMEM;
  } catch (...) {
    return AIMS_ERR_INVALID_ARG;
  }
}

int aims_gpu_wrap_points(int device, void *cuda_stream, const double *lattice, int64_t n_points, double *xyz) {
  if (!lattice || n_points < 0 || (n_points > 0 && !xyz)) return AIMS_ERR_INVALID_ARG;
  Inv3 M;
  for (int i = 0; i < 9; i++) M.a[i] = lattice[i];
  if (!invert3(lattice, M.inv)) return AIMS_ERR_INVALID_ARG;
  if (n_points == 0) return AIMS_OK;
  if (cudaSetDevice(device) != cudaSuccess) return AIMS_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const long long nb = (n_points + 255) / 256;
  k_wrap_points<<<(unsigned)nb, 256, 0, st>>>(M, (long long)n_points, xyz);
  return cudaGetLastError() == cudaSuccess ? AIMS_OK : AIMS_ERR_CUDA;
}

}  // extern "C"
