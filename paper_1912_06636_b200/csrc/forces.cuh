// forces.cuh -- Pulay forces (Eq. 14-18), evaluated batch by batch "alongside
// the density update" (L301-308, L405) on the FP64 tensor pipe.
//
// With the reduced h_KS of this build (local potential v plus the GGA term in its integrated-by-parts form, DESIGN.md
// reading P2) and nabla_at phi_i = -grad phi_i for the functions centred on atom `at`, Eq. 16 and Eq. 18 read on the grid
//   F_at = 2 sum_p sum_{i on at} [ w grad phi_i ]_p X_ip  +  2 sum_p sum_{i on at} [ w Hess phi_i g ]_p T_ip ,
//   X = n_b (v Phi + g.grad Phi) - q_b Phi ,     T = n_b Phi ,
// n_b, q_b = density matrix and energy-weighted density matrix (Eq. 17) restricted to nnz(B).  X and T are the same
// DSYMM-shaped products as the density update (Fig. 6b L359/L370): X is ONE product over K = 2 nnz -- first q_b Phi, then
// the accumulators change sign, then n_b L is added on top -- and T a second one.  The
// epilogue multiplies the accumulator block with the weighted derivative planes written by k_eval<kEvalForce*>, reduces
// over the POINTS of the block (registers, then shuffles over the four lanes of a row) and adds the row sums to a per-CTA
// table of active atoms in shared memory; the CTA finally adds nact x 3 numbers to F with FP64 REDs.
//
// CTA shape, pipeline, operand layouts, block dealing and the D_b gather are those of k_density (density.cuh).
#pragma once
#include "common.cuh"
#include "density.cuh"

namespace aims {

struct FArgs {
  const DItem *items;
  const int *order;                 // launch order: CTA x works on items[order[x]] (NULL: items[x])
  const double *P, *Lp;             // planes Phi and L = v Phi (+ g.grad Phi), density layout
  const double *E[6];               // w d_c Phi (c = x,y,z) and, GGA only, w (Hess Phi g)_c
  const long long *pad_off;         // [n_batches+1] prefix of round_up(nnz,16)*pad8(np)
  long long pad_base;
  const double *D, *Q;              // block-sparse n_ij and q_ij (Q may be NULL: no energy-weighted term)
  double *F;                        // [n_atoms][3]
  int max_nnz_pad;                  // capacity of the fn_info smem array
  int ptab_in_smem;
  double *sigma;                    // STRESS only: [3][3], sigma[l][m] += (1/V) dE/d eps_lm of the launch's batches
  double inv_volume;
};

inline size_t f_smem_bytes(int max_nnz, int max_act, bool ptab_in_smem) {
  size_t s = (size_t)kDStages * kDStage * sizeof(double);
  s += (size_t)(kMaxActive * 3 + 16) * sizeof(double);        // per-CTA force table [slot][3] + stress sums [3][3]
  s += 2 * kDStages * sizeof(unsigned long long);             // full / empty barriers
  if (ptab_in_smem) s += (size_t)max_act * max_act * sizeof(long long);
  s += (size_t)pad8(max_nnz) * sizeof(int) + (size_t)kMaxActive * sizeof(int);
  return s;
}

// STRESS: additionally the Pulay part of the stress tensor (Eq. 20; L299-308; L405 "the Pulay contribution
// to F_at and sigma_lm"): the same integrand weighted with the distance vector to the function's own atom (DESIGN.md reading
// P22),  V sigma_lm = 2 sum_p sum_i (r_p - R_at(i))_m [ ... ]_l .  Written relative to a reference point c of the batch,
//   sum_i sum_p (r_p - c)_m [...]_l  -  sum_slots (R_slot - c)_m sF[slot][l] ,
// the first sum needs no per-atom separation (nine more accumulators per lane, weighted with the lane's two points) and the
// second comes from the CTA's force table; both terms are of the size of the batch, so nothing cancels.
template <bool GGA, bool STRESS, int NMMA>
__device__ __forceinline__ void d_forces_body(const DevSys &S, const BatchLists &L, const FArgs &A, int max_act, const DItem it) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double *sA = reinterpret_cast<double *>(smem_raw);                     // stage s: [k4][tm][4] at sA + s * kDStage
  double *sF = sA + (size_t)kDStages * kDStage;                          // [slot][3]
  double *sG = sF + kMaxActive * 3;                                      // [3][3] (STRESS)
  unsigned long long *s_bar = reinterpret_cast<unsigned long long *>(sG + 16);
  int *sInfo = reinterpret_cast<int *>(s_bar + 2 * kDStages);           // 16-byte aligned; [pad8(max nnz)]
  int *sLd = sInfo + pad8(A.max_nnz_pad);
  long long *sPtab = reinterpret_cast<long long *>(sLd + kMaxActive);

  const int b = it.b;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nnz = L.nnz[b], nact = L.n_act[b];
  const int nnz8 = pad8(nnz), nsub = nnz8 >> 3, nblk = blk_count(nsub);
  const int np = (int)(S.batch_ptr[b + 1] - S.batch_ptr[b]);
  const int np8 = pad8(np);
  const long long boff = A.pad_off[b] - A.pad_base;
  const int p0 = it.p0, npt = it.npt;                    // this CTA's points [p0, p0+npt) of the batch (multiples of 8)
  const int psub = npt >> 3, PB = blk_count(psub);
  constexpr int nmma = NMMA, nprod = (16 - NMMA) * 32;         // MMA warps and producer lanes of this CTA
  const int IB = min(8, nmma / PB);
  const int n_mt = (nblk + IB - 1) / IB;
  const double *sB = sA + IB * 32 * kDKC;
  const int nkc = (nnz8 + kDKC - 1) / kDKC;
  const long long fo = L.fn_off[b], ao = L.act_off[b];
  const long long *gptab = L.ptab + L.ptab_off[b];
  // K segments of the two products: pass 0 (X): [q_b | Phi] then [n_b | L]; pass 1 (T, GGA only): [n_b | Phi]
  constexpr int NPASS = GGA ? 2 : 1;
  const int nseg0 = A.Q ? 2 : 1;

  for (int i = tid; i < nnz8; i += kDThreads) sInfo[i] = i < nnz ? L.fn_info[fo + i] : -1;
  for (int i = tid; i < nact; i += kDThreads) sLd[i] = L.act_ld[ao + i];
  if (A.ptab_in_smem)
    for (int i = tid; i < nact * nact; i += kDThreads) sPtab[i] = gptab[i];
  for (int i = tid; i < kMaxActive * 3 + 16; i += kDThreads) sF[i] = 0.0;
  const long long pbase = S.batch_ptr[b];
  double cref[3] = {0.0, 0.0, 0.0};                      // reference point of the batch (STRESS): its first point
  if (STRESS && np > 0) { cref[0] = S.px[pbase]; cref[1] = S.py[pbase]; cref[2] = S.pz[pbase]; }
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
      for (int pass = 0; pass < NPASS; pass++) {
        const int nseg = pass == 0 ? nseg0 : 1;
#pragma unroll 1
        for (int seg = 0; seg < nseg; seg++) {
          const bool qseg = pass == 0 && seg < nseg - 1;
          const double *M = qseg ? A.Q : A.D;
          const double *gB = ((pass == 0 && !qseg) ? A.Lp : A.P) + boff;
#pragma unroll 1
          for (int kc = 0; kc < nkc; kc++, step++) {
            const int s = step % kDStages;
            if (step >= kDStages) mbar_wait(bar_empty + 8 * s, (unsigned)(step / kDStages - 1) & 1u);
            const int k0 = kc * kDKC;
            if (seg == nseg - 1 && kc == max(nkc - kDPrefetchLead, 0)) {
              // operands of this pass's epilogue (rows [i0, i0+tm) of three derivative planes at the CTA's points)
              const int c0 = i0 >> 4, nch = ((i0 + tm - 1) >> 4) - c0 + 1;
              for (int idx = pl; idx < nch * 3; idx += nprod) {
                const int c = c0 + idx / 3, q = idx % 3;
                bulk_prefetch_l2(A.E[3 * pass + q] + boff + ((long long)c * (np8 >> 2) + (p0 >> 2)) * 64, (unsigned)npt * 128u);
              }
            }
            if (pl == nprod - 1) {
              mbar_expect_tx(bar_full + 8 * s, (unsigned)npt * 128u);
              bulk_g2s(smem_u32(sB + (size_t)s * kDStage), gB + ((long long)kc * (np8 >> 2) + (p0 >> 2)) * 64, (unsigned)npt * 128u,
                       bar_full + 8 * s);
            }
            d_gather_tile(sA + (size_t)s * kDStage, M, i0, tm, k0, nnz, nnz8, nact, sInfo, sLd, ptab, pl, nprod);
            cp_async_mbar_arrive_noinc(bar_full + 8 * s);
          }
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
    double G[STRESS ? 3 : 1][3];                         // sum over rows and points of (r_p - c)_m [...]_l
#pragma unroll
    for (int l = 0; l < (STRESS ? 3 : 1); l++)
#pragma unroll
      for (int m = 0; m < 3; m++) G[l][m] = 0.0;

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
      for (int pass = 0; pass < NPASS; pass++) {
        const int nseg = pass == 0 ? nseg0 : 1;
#pragma unroll 1
        for (int seg = 0; seg < nseg; seg++) {
          d_mma_kloop(blive ? variant : 0, acc, sA + aoffl, sB + boffl, tm, nkc, nnz8, step, bar_full, bar_empty, lane);
          if (seg < nseg - 1) {
            // end of the q_b Phi segment: flip the sign, n_b L is added on top in the next segment (X = n_b L - q_b Phi)
#pragma unroll
            for (int a = 0; a < 4; a++)
#pragma unroll
              for (int c = 0; c < 4; c++) { acc[a][c][0] = -acc[a][c][0]; acc[a][c][1] = -acc[a][c][1]; }
          }
        }
        if (blive) {
          // ---- epilogue of this pass: row sums over the block's points of acc * (weighted derivative plane)
          // two row sub-tiles at a time; per point sub-tile their six loads (L2-prefetched by the producers) are issued
          // before the first FMA
#pragma unroll
          for (int a0 = 0; a0 < 4; a0 += 2) {
            if (a0 < wa) {
              double f[2][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
              const int i_[2] = {ri0 + a0 * 8 + fr, ri0 + min(a0 + 1, wa - 1) * 8 + fr};   // < nnz8: padding rows are zero in the planes
#pragma unroll
              for (int c = 0; c < 4; c++) {
                if (c < wb) {
                  const int p = p0 + ps0 + c * 8 + 2 * fk;           // within the batch (even)
                  double rp[STRESS ? 2 : 1][3];                       // the lane's two points relative to the reference
                  if (STRESS) {
#pragma unroll
                    for (int e = 0; e < 2; e++) {
                      const long long pg = pbase + min(p + e, np - 1);   // padding points: planes are zero there
                      rp[STRESS ? e : 0][0] = S.px[pg] - cref[0]; rp[STRESS ? e : 0][1] = S.py[pg] - cref[1];
                      rp[STRESS ? e : 0][2] = S.pz[pg] - cref[2];
                    }
                  }
                  double2 ev[2][3];
#pragma unroll
                  for (int da = 0; da < 2; da++) {
                    const int i = i_[da];
                    const long long o = boff + (((long long)(i >> 4) * (np8 >> 2) + (p >> 2)) * 16 + (i & 15)) * 4 + (p & 3);
#pragma unroll
                    for (int q = 0; q < 3; q++) ev[da][q] = __ldg(reinterpret_cast<const double2 *>(A.E[3 * pass + q] + o));
                  }
#pragma unroll
                  for (int da = 0; da < 2; da++)
#pragma unroll
                    for (int q = 0; q < 3; q++) {
                      if (!STRESS) {
                        f[da][q] += ev[da][q].x * acc[min(a0 + da, 3)][c][0] + ev[da][q].y * acc[min(a0 + da, 3)][c][1];
                      } else {
                        const double t0 = ev[da][q].x * acc[min(a0 + da, 3)][c][0], t1 = ev[da][q].y * acc[min(a0 + da, 3)][c][1];
                        f[da][q] += t0 + t1;
                        if (a0 + da < wa) {                            // the clamped duplicate row must not count twice
#pragma unroll
                          for (int m = 0; m < 3; m++) G[STRESS ? q : 0][m] += t0 * rp[0][m] + t1 * rp[STRESS ? 1 : 0][m];
                        }
                      }
                    }
                }
              }
#pragma unroll
              for (int da = 0; da < 2; da++) {
                const int fi = sInfo[i_[da]];
#pragma unroll
                for (int q = 0; q < 3; q++) {
                  double v = f[da][q];
                  v += __shfl_xor_sync(0xffffffffu, v, 1);
                  v += __shfl_xor_sync(0xffffffffu, v, 2);
                  if (fk == 0 && fi >= 0 && a0 + da < wa) atomicAdd(sF + (fi >> 16) * 3 + q, v);
                }
              }
            }
          }
        }
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
          for (int c = 0; c < 4; c++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }
      }
    }
    if (STRESS) {
#pragma unroll
      for (int l = 0; l < 3; l++)
#pragma unroll
        for (int m = 0; m < 3; m++) {
          double u = G[STRESS ? l : 0][m];
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) u += __shfl_xor_sync(0xffffffffu, u, o);
          if (lane == 0) atomicAdd(sG + 3 * l + m, u);
        }
    }
  }
  __syncthreads();

  // ---- the CTA's contribution to F: nact x 3 numbers (factor 2 of Eq. 16/18: both index orders of the symmetric sums)
  if (A.F)
    for (int i = tid; i < nact * 3; i += kDThreads) {
      const int s = i / 3, q = i - 3 * s;
      red_add_f64(A.F + (long long)L.act_atom[ao + s] * 3 + q, 2.0 * sF[i]);
    }
  if (STRESS && tid < 9) {
    const int l = tid / 3, m = tid - 3 * l;
    double u = sG[tid];
    for (int s = 0; s < nact; s++) u -= (S.atom_xyz[3 * L.act_atom[ao + s] + m] - cref[m]) * sF[3 * s + l];
    red_add_f64(A.sigma + tid, 2.0 * u * A.inv_volume);
  }
}

template <bool GGA, bool STRESS>
__global__ void __launch_bounds__(kDThreads, 1) k_forces(DevSys S, BatchLists L, FArgs A, int max_act) {
  const DItem it = A.items[A.order ? A.order[blockIdx.x] : blockIdx.x];
  if (d_mma_warps(blk_count(it.npt >> 3)) == 12) d_forces_body<GGA, STRESS, 12>(S, L, A, max_act, it);
  else d_forces_body<GGA, STRESS, 14>(S, L, A, max_act, it);
}

}  // namespace aims
