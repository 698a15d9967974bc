// hamiltonian.cuh -- S2b/S2c/S2d: batch contraction h[B] = K . L (Eq. 25-27) on the FP64 tensor pipe
// (DMMA.8x8x4), fused with the scatter into the atom-pair block-sparse H ("insert_into_h", L327/L342, L385-388).
//
// Operands come from the planes written by k_eval: P = Phi and Q = w v Phi (LDA) or w (v/2 Phi + g.grad Phi) (GGA).
//   LDA : h[B] = P Q^T                 (symmetric; SYRK-shaped, paper: dgmm + syr2k with h phi = v phi)
//   GGA : h[B] = P Q^T + Q P^T         (SYR2K-shaped, as in Fig. 6a)
// Only upper tiles (tj >= ti) of the nnz x nnz batch matrix are computed; on diagonal tiles only 8x8 sub-tiles on or
// above the diagonal.  One CTA (16 warps) per tile of T x T (T <= 128, multiple of 8, balanced per batch); warp
// (wm, wn) owns the 8x8 sub-tiles (mi, ni) with mi = wm mod 4, ni = wn mod 4, so ragged tiles and diagonal tiles stay
// balanced over the four SM sub-partitions.
#pragma once
#include "common.cuh"

namespace aims {

constexpr int kHT = 128;          // max tile edge
constexpr int kHKC = 16;          // points per pipeline stage
constexpr int kHLds = kHKC + 4;   // smem row stride in doubles: (row*20 + k) mod 16 distinct over an 8x4 fragment
constexpr int kHPanel = kHT * kHLds;           // doubles per panel per stage
constexpr int kHCld = kHT + 8;    // row stride of the C staging tile (conflict-free 16-byte fragment stores)
constexpr int kHThreads = 512;

struct HTile { int b, ti, tj, t; };

struct HArgs {
  const HTile *tiles;       // tile list of this launch (already offset)
  const double *P, *Q;      // planes
  const long long *pad_off; // [n_batches+1] prefix of nnz*ld (doubles)
  long long pad_base;
  double *H;                // block-sparse values
};

template <bool GGA>
__host__ __device__ constexpr int h_stages() { return GGA ? 2 : 3; }
template <bool GGA>
constexpr size_t h_smem_bytes() {
  size_t pipe = (size_t)h_stages<GGA>() * (GGA ? 4 : 2) * kHPanel * sizeof(double);
  size_t cst = (size_t)kHT * kHCld * sizeof(double);
  return (pipe > cst ? pipe : cst) + 2 * kHT * sizeof(int) + kMaxActive * sizeof(int);
}

template <bool GGA>
__global__ void __launch_bounds__(kHThreads, 1) k_hamiltonian(DevSys S, BatchLists L, HArgs A) {
  constexpr int NST = h_stages<GGA>();
  constexpr int NPAN = GGA ? 4 : 2;   // panels per stage: P_I, Q_J [, Q_I, P_J]
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *sm = reinterpret_cast<double *>(smem_raw);
  constexpr size_t pipe_d = (size_t)NST * NPAN * kHPanel, cst_d = (size_t)kHT * kHCld;
  int *s_rowinfo = reinterpret_cast<int *>(sm + (pipe_d > cst_d ? pipe_d : cst_d));
  int *s_colinfo = s_rowinfo + kHT;
  int *s_ld = s_colinfo + kHT;

  const HTile tile = A.tiles[blockIdx.x];
  const int b = tile.b, T = tile.t;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wn = warp >> 2, wm = (warp + wn) & 3;   // each SM sub-partition (warp & 3) sees every wm and every wn
  const int nnz = L.nnz[b], nact = L.n_act[b];
  const int np = (int)(S.batch_ptr[b + 1] - S.batch_ptr[b]);
  const int ld = round_up(np, kPadPts);
  const long long boff = A.pad_off[b] - A.pad_base;
  const int i0 = tile.ti * T, j0 = tile.tj * T;
  const int vi = min(T, nnz - i0), vj = min(T, nnz - j0);   // valid rows / cols of this tile
  const bool diag = (tile.ti == tile.tj);
  const long long fo = L.fn_off[b], ao = L.act_off[b];

  // row / column bookkeeping for the scatter
  for (int r = tid; r < kHT; r += kHThreads) {
    s_rowinfo[r] = (r < vi) ? L.fn_info[fo + i0 + r] : 0;
    s_colinfo[r] = (r < vj) ? L.fn_info[fo + j0 + r] : 0;
  }
  for (int s = tid; s < nact; s += kHThreads) s_ld[s] = L.act_ld[ao + s];

  // which of my 4x4 sub-tiles exist
  const int nsi = (vi + 7) >> 3, nsj = (vj + 7) >> 3;
  unsigned amask = 0;
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int c = 0; c < 4; c++) {
      const int mi = wm + 4 * a, ni = wn + 4 * c;
      if (mi < nsi && ni < nsj && (!diag || ni >= mi)) amask |= 1u << (a * 4 + c);
    }
  unsigned rmask = 0, cmask = 0;   // rows a / cols c with any live sub-tile
#pragma unroll
  for (int a = 0; a < 4; a++)
    if (amask >> (a * 4) & 0xFu) rmask |= 1u << a;
#pragma unroll
  for (int c = 0; c < 4; c++)
    if (amask & (0x1111u << c)) cmask |= 1u << c;

  double acc[4][4][2];
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int c = 0; c < 4; c++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }

  // ---- producer: 16-byte cp.async of one K-chunk (kHKC points) of every panel
  const double *gP = A.P + boff, *gQ = A.Q + boff;
  const int nk = ld / kHKC;
  auto load_stage = [&](int stage, int kc) {
    double *base = sm + (size_t)stage * NPAN * kHPanel;
    const int pcol = kc * kHKC;
    // chunk id: 8 chunks of 16 B per row, kHT rows, NPAN panels
    for (int c = tid; c < NPAN * kHT * 8; c += kHThreads) {
      const int pan = c / (kHT * 8), rem = c - pan * (kHT * 8);
      const int r = rem >> 3, ch = rem & 7;
      const bool isI = (pan == 0 || pan == 2);
      const int row = (isI ? i0 : j0) + r;
      const bool ok = r < (isI ? vi : vj);
      const double *plane = (pan == 0 || pan == 3) ? gP : gQ;
      const double *src = plane + (long long)(ok ? row : 0) * ld + pcol + ch * 2;
      cp_async16(smem_u32(base + (size_t)pan * kHPanel + r * kHLds + ch * 2), src, ok ? 16 : 0);
    }
  };

#pragma unroll
  for (int s = 0; s < NST - 1; s++) {
    if (s < nk) load_stage(s, s);
    cp_async_commit();
  }

  const int fr = lane >> 2, fk = lane & 3;
  for (int kc = 0; kc < nk; kc++) {
    cp_async_wait<NST - 2>();
    __syncthreads();
    {  // prefetch chunk kc+NST-1 into the stage freed by the previous iteration
      const int nx = kc + NST - 1;
      if (nx < nk) load_stage(nx % NST, nx);
      cp_async_commit();
    }
    const double *st = sm + (size_t)(kc % NST) * NPAN * kHPanel;
    const double *sPI = st, *sQJ = st + kHPanel, *sQI = st + 2 * kHPanel, *sPJ = st + 3 * kHPanel;
#pragma unroll
    for (int ks = 0; ks < kHKC / 4; ks++) {
      double fa[4], fb[4], ga[4], gb[4];
#pragma unroll
      for (int a = 0; a < 4; a++) {
        const int o = ((wm + 4 * a) * 8 + fr) * kHLds + ks * 4 + fk;
        if (rmask >> a & 1u) { fa[a] = sPI[o]; if (GGA) ga[a] = sQI[o]; }
      }
#pragma unroll
      for (int c = 0; c < 4; c++) {
        const int o = ((wn + 4 * c) * 8 + fr) * kHLds + ks * 4 + fk;
        if (cmask >> c & 1u) { fb[c] = sQJ[o]; if (GGA) gb[c] = sPJ[o]; }
      }
#pragma unroll
      for (int a = 0; a < 4; a++)
#pragma unroll
        for (int c = 0; c < 4; c++)
          if (amask >> (a * 4 + c) & 1u) {
            dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
            if (GGA) dmma8x8x4(acc[a][c][0], acc[a][c][1], ga[a], gb[c]);
          }
    }
  }
  cp_async_wait<0>();
  __syncthreads();

  // ---- epilogue: stage the tile in smem, then add row segments into the block-sparse H (S2d)
  double *sC = sm;
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int c = 0; c < 4; c++)
      if (amask >> (a * 4 + c) & 1u) {
        const int r = (wm + 4 * a) * 8 + fr, cc = (wn + 4 * c) * 8 + 2 * fk;
        *reinterpret_cast<double2 *>(sC + r * kHCld + cc) = make_double2(acc[a][c][0], acc[a][c][1]);
      }
  __syncthreads();
  const long long *ptab = L.ptab + L.ptab_off[b];
  for (int r = warp; r < vi; r += kHThreads / 32) {
    const int ri = s_rowinfo[r];
    const int si = ri >> 16, ai = ri & 0xFFFF;
    for (int c = lane; c < vj; c += 32) {
      if (diag && (c >> 3) < (r >> 3)) continue;            // sub-tile below the diagonal: not computed
      const int ci = s_colinfo[c];
      const int sj = ci >> 16, bj = ci & 0xFFFF;
      if (si > sj) continue;                                // lower atom block (only inside diagonal sub-tiles)
      const long long base = __ldg(ptab + si * nact + sj);
      if (base < 0) continue;                               // atom pair outside the pattern: exact zero
      const double val = sC[r * kHCld + c];
      const int ldb = s_ld[sj];
      red_add_f64(A.H + base + (long long)ai * ldb + bj, val);
      // diagonal atom block holds the full square: mirror unless (c,r) is itself computed in this tile
      if (si == sj && !(diag && (c >> 3) == (r >> 3))) red_add_f64(A.H + base + (long long)bj * ldb + ai, val);
    }
  }
}

}  // namespace aims
