// hessian.cuh -- Hessian of the density ("the Hessian matrix of the density ... six
// components, and each component has the same cost as the evaluation of n(r) itself"), batch by batch on the FP64 tensor
// pipe.  For symmetric n_ij restricted to nnz(B):
//   d_c d_e n_p = 2 sum_i (d_c d_e Phi)_ip T_ip  +  2 sum_i (d_c Phi)_ip (U_e)_ip ,   T = n_b Phi ,  U_e = n_b (d_e Phi) ,
// i.e. four DSYMM-shaped products per M-tile (B operand Phi, d_x Phi, d_y Phi, d_z Phi; the same D_b tile gather), each
// followed by an epilogue that multiplies the accumulator block with derivative planes written by k_eval<kEvalHess> and
// reduces over the ROWS of the block (shuffles), exactly as k_density does for n and grad n:
//   pass 0 (T)   : the six Hessian planes            -> xx, yy, zz, xy, xz, yz
//   pass 1 (U_x) : d_x Phi                           -> xx
//   pass 2 (U_y) : d_x Phi, d_y Phi                  -> xy, yy
//   pass 3 (U_z) : d_x Phi, d_y Phi, d_z Phi         -> xz, yz, zz
// (sum_ij d_c Phi_i n_ij d_e Phi_j is symmetric in (c, e) because n_ij is.)  Partial sums per row block live in shared
// memory, one owner warp per (row block, column): no atomics, bitwise reproducible.
// CTA shape, pipeline, operand layouts, block dealing and the D_b gather are those of k_density (density.cuh).
#pragma once
#include "common.cuh"
#include "density.cuh"

namespace aims {

struct XArgs {
  const DItem *items;
  const int *order;                 // launch order: CTA x works on items[order[x]] (NULL: items[x])
  const double *PL[10];             // planes Phi, d_x, d_y, d_z Phi, then d_c d_e Phi (xx, yy, zz, xy, xz, yz); density layout
  const long long *pad_off;         // [n_batches+1] prefix of round_up(nnz,16)*pad8(np)
  long long pad_base;
  const double *D;                  // block-sparse n_ij
  double *hn;                       // [6][n_points]
  long long n_points;
  int max_nnz_pad;
  int ptab_in_smem;
};

inline size_t x_smem_bytes(int max_nnz, int max_act, bool ptab_in_smem) {
  size_t s = (size_t)kDStages * kDStage * sizeof(double);
  s += (size_t)6 * kDPartCols * sizeof(double);               // part[ib][component][col of the CTA]
  s += 2 * kDStages * sizeof(unsigned long long);
  if (ptab_in_smem) s += (size_t)max_act * max_act * sizeof(long long);
  s += (size_t)pad8(max_nnz) * sizeof(int) + (size_t)kMaxActive * sizeof(int);
  return s;
}

// epilogue of one pass: NT terms; term t multiplies the accumulators with plane pl[t] and adds to component comp[t]
template <int NT>
__device__ __forceinline__ void x_epilogue(const double (&acc)[4][4][2], const XArgs &A, const int (&pl)[6], const int (&comp)[6],
                                           double *sPart, long long boff, int np8, int p0, int ps0, int ri0, int wa, int wb, int ib,
                                           int npt, int fr, int fk) {
#pragma unroll
  for (int c = 0; c < 4; c++) {
    if (c < wb) {
      const int col = ps0 + c * 8 + 2 * fk;            // within the CTA's point range (even)
      const int p = p0 + col;                          // within the batch
      double s[NT][2];
#pragma unroll
      for (int t = 0; t < NT; t++) { s[t][0] = 0.0; s[t][1] = 0.0; }
#pragma unroll
      for (int a = 0; a < 4; a++) {
        if (a < wa) {
          const int i = ri0 + a * 8 + fr;              // < nnz8: padding rows are zero in the planes
          const long long o = boff + (((long long)(i >> 4) * (np8 >> 2) + (p >> 2)) * 16 + (i & 15)) * 4 + (p & 3);
          double2 ev[NT];
#pragma unroll
          for (int t = 0; t < NT; t++) ev[t] = __ldg(reinterpret_cast<const double2 *>(A.PL[pl[t]] + o));
#pragma unroll
          for (int t = 0; t < NT; t++) { s[t][0] += ev[t].x * acc[a][c][0]; s[t][1] += ev[t].y * acc[a][c][1]; }
        }
      }
#pragma unroll
      for (int t = 0; t < NT; t++)
#pragma unroll
        for (int e = 0; e < 2; e++) {
          double v = s[t][e];
          v += __shfl_xor_sync(0xffffffffu, v, 4); v += __shfl_xor_sync(0xffffffffu, v, 8); v += __shfl_xor_sync(0xffffffffu, v, 16);
          s[t][e] = v;
        }
      if (fr == 0) {   // lanes 0..3 own columns 2*fk, 2*fk+1; (ib, column) has exactly one owner warp -> no race
#pragma unroll
        for (int t = 0; t < NT; t++) {
          double *pp = sPart + (ib * 6 + comp[t]) * npt + col;
          pp[0] += s[t][0]; pp[1] += s[t][1];
        }
      }
    }
  }
}

template <int NMMA>
__device__ __forceinline__ void d_hessian_body(const DevSys &S, const BatchLists &L, const XArgs &A, int max_act, const DItem it) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double *sA = reinterpret_cast<double *>(smem_raw);                     // stage s: [k4][tm][4] at sA + s * kDStage
  double *sPart = sA + (size_t)kDStages * kDStage;                       // [ib][component][col]
  unsigned long long *s_bar = reinterpret_cast<unsigned long long *>(sPart + 6 * kDPartCols);
  int *sInfo = reinterpret_cast<int *>(s_bar + 2 * kDStages);
  int *sLd = sInfo + pad8(A.max_nnz_pad);
  long long *sPtab = reinterpret_cast<long long *>(sLd + kMaxActive);

  const int b = it.b;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nnz = L.nnz[b], nact = L.n_act[b];
  const int nnz8 = pad8(nnz), nsub = nnz8 >> 3, nblk = blk_count(nsub);
  const long long pbase = S.batch_ptr[b];
  const int np = (int)(S.batch_ptr[b + 1] - pbase);
  const int np8 = pad8(np);
  const long long boff = A.pad_off[b] - A.pad_base;
  const int p0 = it.p0, npt = it.npt;
  const int psub = npt >> 3, PB = blk_count(psub);
  constexpr int nmma = NMMA, nprod = (16 - NMMA) * 32;         // MMA warps and producer lanes of this CTA
  const int IB = min(8, nmma / PB);
  const int n_mt = (nblk + IB - 1) / IB;
  const double *sB = sA + IB * 32 * kDKC;
  const int nkc = (nnz8 + kDKC - 1) / kDKC;
  const long long fo = L.fn_off[b], ao = L.act_off[b];
  const long long *gptab = L.ptab + L.ptab_off[b];

  for (int i = tid; i < nnz8; i += kDThreads) sInfo[i] = i < nnz ? L.fn_info[fo + i] : -1;
  for (int i = tid; i < nact; i += kDThreads) sLd[i] = L.act_ld[ao + i];
  if (A.ptab_in_smem)
    for (int i = tid; i < nact * nact; i += kDThreads) sPtab[i] = gptab[i];
  for (int i = tid; i < 6 * kDPartCols; i += kDThreads) sPart[i] = 0.0;
  const unsigned bar_full = smem_u32(s_bar), bar_empty = bar_full + 8 * kDStages;
  __shared__ int s_map[kDMmaWarps];
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kDStages; s++) {
      mbar_init(bar_full + 8 * s, (unsigned)nprod + 1u);
      mbar_init(bar_empty + 8 * s, (unsigned)nmma);
    }
    mbar_fence_init();
    d_deal_blocks(s_map, PB, IB, psub, nmma);
  }
  __syncthreads();
  const long long *ptab = A.ptab_in_smem ? sPtab : gptab;

  if (warp >= nmma) {
    // =========================================================================== producers
    const int pl = tid - nmma * 32;
    int step = 0;
#pragma unroll 1
    for (int mt = 0; mt < n_mt; mt++) {
      const int bi0 = mt * IB, bi1 = min(bi0 + IB, nblk);
      const int i0 = blk_start(bi0, nsub, nblk), tm = blk_start(bi1, nsub, nblk) - i0;
#pragma unroll 1
      for (int pass = 0; pass < 4; pass++) {
        const double *gB = A.PL[pass] + boff;            // B operand of the pass: Phi, d_x Phi, d_y Phi, d_z Phi
#pragma unroll 1
        for (int kc = 0; kc < nkc; kc++, step++) {
          const int s = step % kDStages;
          if (step >= kDStages) mbar_wait(bar_empty + 8 * s, (unsigned)(step / kDStages - 1) & 1u);
          const int k0 = kc * kDKC;
          if (kc == max(nkc - kDPrefetchLead, 0)) {
            // operands of this pass's epilogue: rows [i0, i0+tm) of the six Hessian planes (pass 0) or of d_x..d_e Phi
            const int c0 = i0 >> 4, nch = ((i0 + tm - 1) >> 4) - c0 + 1;
            const int npl = pass == 0 ? 6 : pass, pl0 = pass == 0 ? 4 : 1;
            for (int idx = pl; idx < nch * npl; idx += nprod) {
              const int c = c0 + idx / npl, q = idx % npl;
              bulk_prefetch_l2(A.PL[pl0 + q] + boff + ((long long)c * (np8 >> 2) + (p0 >> 2)) * 64, (unsigned)npt * 128u);
            }
          }
          if (pl == nprod - 1) {
            mbar_expect_tx(bar_full + 8 * s, (unsigned)npt * 128u);
            bulk_g2s(smem_u32(sB + (size_t)s * kDStage), gB + ((long long)kc * (np8 >> 2) + (p0 >> 2)) * 64, (unsigned)npt * 128u,
                     bar_full + 8 * s);
          }
          d_gather_tile(sA + (size_t)s * kDStage, A.D, i0, tm, k0, nnz, nnz8, nact, sInfo, sLd, ptab, pl, nprod);
          cp_async_mbar_arrive_noinc(bar_full + 8 * s);
        }
      }
    }
  } else {
    // =========================================================================== MMA warps
    const int wmap = s_map[warp];
    const bool wlive = wmap >= 0;
    const int pb = wmap & 0xFF, ib = wlive ? (wmap >> 8) : 0;
    const int ps0 = wlive ? blk_start(pb, psub, PB) : 0;
    const int wb = wlive ? (blk_start(pb + 1, psub, PB) - ps0) >> 3 : 0;
    const int fr = lane >> 2, fk = lane & 3;
    const int boffl = (ps0 >> 2) * (kDKC * 4) + (fr >> 2) * (kDKC * 4) + fk * 4 + (fr & 3);
    double acc[4][4][2];
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
      for (int c = 0; c < 4; c++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }

    int step = 0;
#pragma unroll 1
    for (int mt = 0; mt < n_mt; mt++) {
      const int bi0 = mt * IB, bi1 = min(bi0 + IB, nblk);
      const int i0 = blk_start(bi0, nsub, nblk), tm = blk_start(bi1, nsub, nblk) - i0;
      const int bi = bi0 + ib;
      const bool blive = wlive && bi < bi1;
      int wa = 0, ri0 = 0;
      if (blive) { ri0 = blk_start(bi, nsub, nblk); wa = (blk_start(bi + 1, nsub, nblk) - ri0) >> 3; }
      const int variant = wa * 4 + wb;
      const int aoffl = (ri0 - i0) * 4 + lane;
#pragma unroll 1
      for (int pass = 0; pass < 4; pass++) {
        d_mma_kloop(blive ? variant : 0, acc, sA + aoffl, sB + boffl, tm, nkc, nnz8, step, bar_full, bar_empty, lane);
        if (blive) {
          // plane and output component of every term of the pass (see the table at the top of the file)
          if (pass == 0) {
            const int pl_[6] = {4, 5, 6, 7, 8, 9}, cm_[6] = {0, 1, 2, 3, 4, 5};
            x_epilogue<6>(acc, A, pl_, cm_, sPart, boff, np8, p0, ps0, ri0, wa, wb, ib, npt, fr, fk);
          } else if (pass == 1) {
            const int pl_[6] = {1, 0, 0, 0, 0, 0}, cm_[6] = {0, 0, 0, 0, 0, 0};
            x_epilogue<1>(acc, A, pl_, cm_, sPart, boff, np8, p0, ps0, ri0, wa, wb, ib, npt, fr, fk);
          } else if (pass == 2) {
            const int pl_[6] = {1, 2, 0, 0, 0, 0}, cm_[6] = {3, 1, 0, 0, 0, 0};
            x_epilogue<2>(acc, A, pl_, cm_, sPart, boff, np8, p0, ps0, ri0, wa, wb, ib, npt, fr, fk);
          } else {
            const int pl_[6] = {1, 2, 3, 0, 0, 0}, cm_[6] = {4, 5, 2, 0, 0, 0};
            x_epilogue<3>(acc, A, pl_, cm_, sPart, boff, np8, p0, ps0, ri0, wa, wb, ib, npt, fr, fk);
          }
        }
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
          for (int c = 0; c < 4; c++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }
      }
    }
  }
  __syncthreads();

  // ---- store: the mapping to the global point array is the identity on the batch's contiguous range
  for (int col = tid; col < npt; col += kDThreads) {
    const int p = p0 + col;
    if (p >= np) continue;
#pragma unroll
    for (int k = 0; k < 6; k++) {
      double u = 0.0;
      for (int m = 0; m < IB; m++) u += sPart[(m * 6 + k) * npt + col];
      A.hn[(long long)k * A.n_points + pbase + p] = 2.0 * u;
    }
  }
}

__global__ void __launch_bounds__(kDThreads, 1) k_density_hessian(DevSys S, BatchLists L, XArgs A, int max_act) {
  const DItem it = A.items[A.order ? A.order[blockIdx.x] : blockIdx.x];
  if (d_mma_warps(blk_count(it.npt >> 3)) == 12) d_hessian_body<12>(S, L, A, max_act, it);
  else d_hessian_body<14>(S, L, A, max_act, it);
}

}  // namespace aims
