// density.cuh -- S3a-S3d: density update n(r) = sum_ij phi_i n_ij phi_j (Eq. 3) per batch as
//   temp = D_b . Phi  (DSYMM of Fig. 6b, L359/L370)  then  n_p = sum_i Phi_ip temp_ip  (L360/L371),
//   grad n_p = 2 sum_i gradPhi_ip temp_ip  (D symmetric; L67, L93-95),
// on the FP64 tensor pipe (DMMA.8x8x4).  D_b ("calculate_density_mat", L314/L357) is never materialised: its tiles are
// gathered straight from the block-sparse D into shared memory with 8-byte cp.async.
//
// One CTA (16 warps) per (batch, point tile of <= 208 points).  It walks the rows of temp in tiles of 64; for each row
// tile the K loop runs over all nnz functions in chunks of 16.  After a row tile its 64 x np accumulators are
// multiplied with Phi (and grad Phi) and reduced over rows with warp shuffles into per-warp-row partial sums in
// shared memory; the final sums are stored once, without atomics (deterministic).
#pragma once
#include "common.cuh"

namespace aims {

constexpr int kDTM = 64;            // rows of temp per row tile
constexpr int kDTN = 208;           // max points per point tile (26 sub-tiles of 8)
constexpr int kDKC = 16;            // K chunk (functions j) per stage
constexpr int kDAld = kDKC + 4;     // smem stride of the D tile rows
constexpr int kDBld = kDTN + 4;     // smem stride of the Phi tile rows ((k*212 + p) mod 16 distinct over a fragment)
constexpr int kDStages = 3;
constexpr int kDThreads = 512;
constexpr int kDNsub = 7;           // n sub-tiles per warp: ceil(26 / 4)

struct DItem { int b, p0, npt, pad; };

struct DArgs {
  const DItem *items;
  const double *P;                  // Phi plane
  const double *G[3];               // gradient planes (GRAD only)
  const long long *pad_off;
  long long pad_base;
  const double *D;                  // block-sparse density matrix
  double *n, *gn;                   // outputs [n_points], [3][n_points]
  long long n_points;
  int max_nnz_pad;                  // capacity of the fn_info smem array
};

inline size_t d_smem_bytes(int max_nnz, int max_act) {
  size_t s = (size_t)kDStages * (kDTM * kDAld + kDKC * kDBld) * sizeof(double);
  s += (size_t)4 * 4 * kDTN * sizeof(double);                 // part[wm][q][col]
  s += (size_t)max_act * max_act * sizeof(long long);         // ptab
  s += (size_t)round_up(max_nnz, 4) * sizeof(int) + (size_t)kMaxActive * sizeof(int);
  return s;
}

template <bool GRAD>
__global__ void __launch_bounds__(kDThreads, 1) k_density(DevSys S, BatchLists L, DArgs A, int max_act) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *sA = reinterpret_cast<double *>(smem_raw);                     // [stage][64][20]
  double *sB = sA + (size_t)kDStages * kDTM * kDAld;                     // [stage][16][212]
  double *sPart = sB + (size_t)kDStages * kDKC * kDBld;                  // [4][4][208]
  long long *sPtab = reinterpret_cast<long long *>(sPart + 4 * 4 * kDTN);
  int *sInfo = reinterpret_cast<int *>(sPtab + (size_t)max_act * max_act);
  int *sLd = sInfo + round_up(A.max_nnz_pad, 4);

  const DItem it = A.items[blockIdx.x];
  const int b = it.b;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wn = warp >> 2, wm = (warp + wn) & 3;
  const int nnz = L.nnz[b], nact = L.n_act[b];
  const long long pbase = S.batch_ptr[b];
  const int np = (int)(S.batch_ptr[b + 1] - pbase);
  const int ld = round_up(np, kPadPts);
  const long long boff = A.pad_off[b] - A.pad_base;
  const int p0 = it.p0, npt = it.npt;                    // this CTA's points [p0, p0+npt) of the batch
  const int nsn = (npt + 7) >> 3;                        // live n sub-tiles
  const long long fo = L.fn_off[b], ao = L.act_off[b];

  for (int i = tid; i < nnz; i += kDThreads) sInfo[i] = L.fn_info[fo + i];
  for (int i = tid; i < nact; i += kDThreads) sLd[i] = L.act_ld[ao + i];
  for (int i = tid; i < nact * nact; i += kDThreads) sPtab[i] = L.ptab[L.ptab_off[b] + i];
  for (int i = tid; i < 4 * 4 * kDTN; i += kDThreads) sPart[i] = 0.0;
  __syncthreads();

  const double *gP = A.P + boff;
  const int nk = (nnz + kDKC - 1) / kDKC;                // K chunks per row tile
  const int nrt = (nnz + kDTM - 1) / kDTM;               // row tiles
  const int nsteps = nk * nrt;

  // ---- producer
  auto load_step = [&](int stage, int step) {
    const int rt = step / nk, kc = step - rt * nk;
    const int k0 = kc * kDKC;
    // A: D_b[rt*64 + r][k0 + k], two elements per thread, gathered from the block pattern
    double *dA = sA + (size_t)stage * kDTM * kDAld;
#pragma unroll
    for (int h = 0; h < (kDTM * kDKC) / kDThreads; h++) {
      const int e = tid + h * kDThreads;
      const int r = e >> 4, k = e & 15;
      const int i = rt * kDTM + r, j = k0 + k;
      const double *src = A.D;
      int bytes = 0;
      if (i < nnz && j < nnz) {
        const int fi = sInfo[i], fj = sInfo[j];
        const int si = fi >> 16, sj = fj >> 16, ai = fi & 0xFFFF, bj = fj & 0xFFFF;
        const long long base = sPtab[si * nact + sj];
        if (base >= 0) {
          src = (si <= sj) ? A.D + base + (long long)ai * sLd[sj] + bj     // stored block (si,sj): row ai, col bj
                           : A.D + base + (long long)bj * sLd[si] + ai;    // stored block (sj,si): transposed read
          bytes = 8;
        }
      }
      cp_async8(smem_u32(dA + r * kDAld + k), src, bytes);
    }
    // B: Phi[k0 + k][p0 .. p0+npt), 16-byte chunks
    double *dB = sB + (size_t)stage * kDKC * kDBld;
    const int nch = (npt + 1) >> 1;                      // chunks per row (npt even except possibly never: ld is even)
    for (int c = tid; c < kDKC * nch; c += kDThreads) {
      const int k = c / nch, ch = c - k * nch;
      const int j = k0 + k;
      const bool ok = j < nnz;
      const double *src = gP + (long long)(ok ? j : 0) * ld + p0 + ch * 2;
      cp_async16(smem_u32(dB + k * kDBld + ch * 2), src, ok ? 16 : 0);
    }
  };

  double acc[2][kDNsub][2];
#pragma unroll
  for (int a = 0; a < 2; a++)
#pragma unroll
    for (int c = 0; c < kDNsub; c++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }

#pragma unroll
  for (int s = 0; s < kDStages - 1; s++) {
    if (s < nsteps) load_step(s, s);
    cp_async_commit();
  }

  const int fr = lane >> 2, fk = lane & 3;
  for (int step = 0; step < nsteps; step++) {
    cp_async_wait<kDStages - 2>();
    __syncthreads();
    {
      const int nx = step + kDStages - 1;
      if (nx < nsteps) load_step(nx % kDStages, nx);
      cp_async_commit();
    }
    const int rt = step / nk, kc = step - rt * nk;
    const double *tA = sA + (size_t)(step % kDStages) * kDTM * kDAld;
    const double *tB = sB + (size_t)(step % kDStages) * kDKC * kDBld;
    const int rows_left = nnz - rt * kDTM;               // live rows in this row tile
#pragma unroll
    for (int ks = 0; ks < kDKC / 4; ks++) {
      double fa[2], fb[kDNsub];
#pragma unroll
      for (int a = 0; a < 2; a++) fa[a] = tA[((wm + 4 * a) * 8 + fr) * kDAld + ks * 4 + fk];
#pragma unroll
      for (int c = 0; c < kDNsub; c++)
        if (wn + 4 * c < nsn) fb[c] = tB[(ks * 4 + fk) * kDBld + (wn + 4 * c) * 8 + fr];
#pragma unroll
      for (int a = 0; a < 2; a++)
        if ((wm + 4 * a) * 8 < rows_left)
#pragma unroll
          for (int c = 0; c < kDNsub; c++)
            if (wn + 4 * c < nsn) dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
    }

    if (kc == nk - 1) {
      // ---- row-tile epilogue: n_p += sum_i Phi_ip temp_ip (and gradient), rows reduced by shuffles
#pragma unroll
      for (int c = 0; c < kDNsub; c++) {
        if (wn + 4 * c < nsn) {
          const int col = (wn + 4 * c) * 8 + 2 * fk;       // within the point tile
          double sn[2] = {0.0, 0.0}, sg[3][2] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
          for (int a = 0; a < 2; a++) {
            const int i = rt * kDTM + (wm + 4 * a) * 8 + fr;
            if (i < nnz) {
              const long long o = (long long)i * ld + p0 + col;
              const double2 ph = *reinterpret_cast<const double2 *>(gP + o);
              sn[0] += ph.x * acc[a][c][0];
              sn[1] += ph.y * acc[a][c][1];
              if (GRAD)
#pragma unroll
                for (int q = 0; q < 3; q++) {
                  const double2 gq = *reinterpret_cast<const double2 *>(A.G[q] + boff + o);
                  sg[q][0] += gq.x * acc[a][c][0];
                  sg[q][1] += gq.y * acc[a][c][1];
                }
            }
          }
#pragma unroll
          for (int e = 0; e < 2; e++) {
            double v = sn[e];
            v += __shfl_xor_sync(0xffffffffu, v, 4); v += __shfl_xor_sync(0xffffffffu, v, 8); v += __shfl_xor_sync(0xffffffffu, v, 16);
            sn[e] = v;
            if (GRAD)
#pragma unroll
              for (int q = 0; q < 3; q++) {
                double u = sg[q][e];
                u += __shfl_xor_sync(0xffffffffu, u, 4); u += __shfl_xor_sync(0xffffffffu, u, 8); u += __shfl_xor_sync(0xffffffffu, u, 16);
                sg[q][e] = u;
              }
          }
          if (fr == 0) {   // lanes 0..3 own columns 2*fk, 2*fk+1; (wm, column) has exactly one owner warp -> no race
            double *pp = sPart + (size_t)(wm * 4) * kDTN + col;
            pp[0] += sn[0]; pp[1] += sn[1];
            if (GRAD)
#pragma unroll
              for (int q = 0; q < 3; q++) { pp[(q + 1) * kDTN] += sg[q][0]; pp[(q + 1) * kDTN + 1] += sg[q][1]; }
          }
        }
#pragma unroll
        for (int a = 0; a < 2; a++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }
      }
    }
  }
  cp_async_wait<0>();
  __syncthreads();

  // ---- S3d: store (mapping to the global point array is the identity on the batch's contiguous range)
  for (int col = tid; col < npt; col += kDThreads) {
    const int p = p0 + col;
    if (p >= np) continue;
    double v = 0.0;
#pragma unroll
    for (int m = 0; m < 4; m++) v += sPart[(size_t)(m * 4) * kDTN + col];
    A.n[pbase + p] = v;
    if (GRAD)
#pragma unroll
      for (int q = 0; q < 3; q++) {
        double u = 0.0;
#pragma unroll
        for (int m = 0; m < 4; m++) u += sPart[(size_t)(m * 4 + q + 1) * kDTN + col];
        A.gn[(long long)q * A.n_points + pbase + p] = 2.0 * u;
      }
  }
}

}  // namespace aims
