// hamiltonian.cuh -- S2b/S2c/S2d: batch contraction h[B] = K . L (Eq. 25-27) on the FP64 tensor pipe
// (DMMA.8x8x4), fused with the scatter into the atom-pair block-sparse H ("insert_into_h", L327/L342, L385-388).
//
// Operands come from the planes written by k_eval (k4 layout, common.cuh): P = Phi and Q = w v Phi (LDA) or
// w (v/2 Phi + g.grad Phi) (GGA).
//   LDA : h[B] = P Q^T                 (symmetric; SYRK-shaped, paper: dgmm + syr2k with h phi = v phi)
//   GGA : h[B] = P Q^T + Q P^T         (SYR2K-shaped, as in Fig. 6a)
//
// Decomposition.  The nnz8 = pad8(nnz) rows of a batch are cut into nblk = ceil(nnz8/32) blocks of 3 or 4 sub-tiles of 8
// rows (no padding beyond the multiple of 8).  Only blocks (bi, bj >= bi) are computed, one warp per block, and on a
// diagonal block only the sub-tiles on or above the diagonal.  A CTA (8 warps) owns an I panel of up to 4 blocks and a
// J panel of up to 2 blocks; two CTAs are resident per SM so that one CTA's scatter epilogue overlaps the other's main
// loop.  B200 measurements behind this shape: a predicated-off DMMA still occupies the pipe
// for its full 16 cycles, so every DMMA here sits in straight-line code selected by warp-uniform branches (one
// template instance per block shape); and one warp per SM sub-partition already sustains 95 % of the DMMA peak, so
// idle warps of ragged or diagonal tiles cost nothing while the co-resident CTA has work.
//
// Pipeline: 3 stages of 8 points; one elected lane issues one bulk async copy (UBLKCP) per panel and 4-point group -- in
// the k4 layout a panel's rows of one group are one contiguous segment -- completing on the stage's "full" mbarrier;
// warps release a stage on its "empty" mbarrier.  There is no CTA-wide barrier after the set-up, so warps of different
// block shapes drift freely and each starts its scatter epilogue (private staging strip) as soon as its block is done.
#pragma once
#include "common.cuh"

namespace aims {

#ifndef AIMS_H_IB
#define AIMS_H_IB 4               // blocks of the I panel: 4 (8 warps, 2 CTAs per SM) or 2 (4 warps, 4 CTAs per SM; profiles/r02_kernel_experiments.md)
#endif
constexpr int kHIB = AIMS_H_IB, kHJB = 2; // blocks per panel
constexpr int kHI = 32 * kHIB;    // max rows of the I panel
constexpr int kHJ = 32 * kHJB;    // max rows of the J panel
constexpr int kHWarps = kHIB * kHJB;      // one warp per block of a full tile
#ifndef AIMS_H_STAGES
#define AIMS_H_STAGES 3
#endif
#ifndef AIMS_H_STRIP_ROWS
#define AIMS_H_STRIP_ROWS 8           // rows of a warp's staging strip: 8, or 4 (two passes per sub-tile row; frees shared memory for a 4th stage)
#endif
constexpr int kHStages = AIMS_H_STAGES;
constexpr int kHStripRows = AIMS_H_STRIP_ROWS;
constexpr int kHThreads = 32 * kHWarps;
constexpr int kHCtasPerSm = 16 / kHWarps;
constexpr int kHStripLd = 40;     // row stride of a warp's 8-row staging strip (conflict-free 16-byte stores)

struct HTile { int b; short ti, tj; };

struct HArgs {
  const HTile *tiles;       // tile list of this launch (already offset)
  const double *P, *Q;      // planes
  const long long *pad_off; // [n_batches+1] prefix of pad8(nnz)*round_up(np, GGA ? 8 : 16) (doubles)
  long long pad_base;
  double *H;                // block-sparse values
  int pmul;                 // planes hold pmul x the (padded) points of a batch: 1, or 3 for the stacked gradient planes of the tau matrix
  // ordered scatter (deterministic mode): CTAs take tiles from `ticket` in list order (sorted by batch)
  // and a tile of batch b adds to H only after `done` says that every tile of the batches before b has finished adding
  int det;
  unsigned *ticket, *done;
  const long long *tile_off;   // [n_batches+1] first tile of every batch (context-wide numbering)
  long long tile_base;         // tile_off of the launch's first batch
};

// first row of block k when nsub sub-tiles of 8 rows are cut into nblk blocks (sizes differ by at most one sub-tile)
__host__ __device__ inline int blk_start(int k, int nsub, int nblk) { return (int)((unsigned)(k * nsub) / (unsigned)nblk) * 8; }
__host__ __device__ inline int blk_count(int nsub) { return (nsub + 3) >> 2; }

template <bool GGA>
__host__ __device__ constexpr int h_group_doubles() { return (kHI + kHJ) * 4 * (GGA ? 2 : 1); }
template <bool GGA>
__host__ __device__ constexpr int h_stage_groups() { return GGA ? 2 : 4; }   // 4-point groups per stage: 8 / 16 points
template <bool GGA>
__host__ __device__ constexpr int h_stage_doubles() { return h_stage_groups<GGA>() * h_group_doubles<GGA>(); }
template <bool GGA>
constexpr size_t h_smem_bytes() {
  return (size_t)kHStages * h_stage_doubles<GGA>() * sizeof(double) + (size_t)kHWarps * kHStripRows * kHStripLd * sizeof(double) +
         2 * kHStages * sizeof(unsigned long long) + (kHI + kHJ + kMaxActive) * sizeof(int);
}

// The whole point loop of one warp block of (8 WA) x (8 WB) outputs as ONE instruction stream of straight-line,
// unpredicated DMMAs.  A stage holds two 4-point groups; per group LDA has one product step (P_I Q_J^T), GGA two
// (P_I Q_J^T, then Q_I P_J^T).  Operand fragments are reloaded in place while the DMMAs of the current step are issued
// (an A fragment is dead after its row, a B fragment after the last row that uses it; on a diagonal block row a uses
// only columns c >= a, so B fragment a dies with row a), and the reloads of a stage's last step already fetch the first
// step of the NEXT stage, whose "full" barrier is waited for after the first row of DMMAs is in the pipe (see
// density.cuh: d_mma_kloop_t for the measurements behind this).
// refill(q): called by lane 0 after chunk q was released -- the kernel's rotating refill duty.
template <int WA, int WB, bool DIAG, bool GGA, class Refill>
__device__ __forceinline__ void h_mma_loop_t(double (&acc)[4][4][2], const double *sm, int aoff, int boff, int nchunk,
                                             unsigned bar_full, unsigned bar_empty, int lane, Refill &&refill) {
  constexpr int NST = kHStages;
  constexpr int GW = h_group_doubles<GGA>(), SW = h_stage_doubles<GGA>();
  constexpr int NU = 4;                                                 // product steps per stage (LDA: 4 groups x 1, GGA: 2 x 2)
  // fragment bases of step u inside a stage
  auto a_base = [&](const double *st, int u) {
    return st + (GGA ? (u >> 1) : u) * GW + ((GGA && (u & 1)) ? (kHI + kHJ) * 4 : 0) + aoff;
  };
  auto b_base = [&](const double *st, int u) {
    return st + (GGA ? (u >> 1) : u) * GW + ((GGA && (u & 1)) ? (2 * kHI + kHJ) * 4 : kHI * 4) + boff;
  };
  mbar_wait(bar_full, 0u);
  const double *st = sm;
  double fa[WA], fb[WB];
  {
    const double *a0 = a_base(st, 0), *b0 = b_base(st, 0);
#pragma unroll
    for (int a = 0; a < WA; a++) fa[a] = a0[a * 32];
#pragma unroll
    for (int c = 0; c < WB; c++) fb[c] = b0[c * 32];
  }
#pragma unroll 1
  for (int q = 0; q < nchunk; q++) {
    const int s = q % NST;
    const double *st1 = st;
#pragma unroll
    for (int u = 0; u < NU; u++) {
      const double *a1, *b1;
      // row 0 first, then (last step of the stage) make sure the next stage has landed before reloading from it
#pragma unroll
      for (int c = 0; c < WB; c++) dmma8x8x4(acc[0][c][0], acc[0][c][1], fa[0], fb[c]);
      if (u + 1 < NU) {
        a1 = a_base(st, u + 1); b1 = b_base(st, u + 1);
      } else {
        if (q + 1 < nchunk) {
          const int s1 = (q + 1) % NST;
          mbar_wait(bar_full + 8 * s1, (unsigned)((q + 1) / NST) & 1u);
          st1 = sm + (size_t)s1 * SW;
        }
        a1 = a_base(st1, 0); b1 = b_base(st1, 0);                       // no next chunk: harmless reload of this stage
      }
      fa[0] = a1[0];
      if (DIAG || WA == 1) fb[0] = b1[0];
#pragma unroll
      for (int a = 1; a < WA; a++) {
#pragma unroll
        for (int c = 0; c < WB; c++)
          if (!DIAG || c >= a) {
            dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
            if (!DIAG && a == WA - 1) fb[c] = b1[c * 32];
          }
        fa[a] = a1[a * 32];
        if (DIAG) fb[a] = b1[a * 32];
      }
      if (!DIAG && WA == 1) {
#pragma unroll
        for (int c = 1; c < WB; c++) fb[c] = b1[c * 32];
      }
    }
    st = st1;
    __syncwarp();
    if (lane == 0) {
      mbar_arrive(bar_empty + 8 * s);                     // every fragment of stage s is in registers
      refill(q);
    }
    __syncwarp();
  }
}

template <bool GGA, class Refill>
__device__ __forceinline__ void h_mma_loop(int variant, double (&acc)[4][4][2], const double *sm, int aoff, int boff,
                                           int nchunk, unsigned bar_full, unsigned bar_empty, int lane, Refill &&refill) {
#define AIMS_H_CASE(WA, WB, DG)                                                                              \
  case (WA * 4 + WB) * 2 + DG:                                                                               \
    h_mma_loop_t<WA, WB, DG != 0, GGA>(acc, sm, aoff, boff, nchunk, bar_full, bar_empty, lane, refill);     \
    break;
  switch (variant) {
    AIMS_H_CASE(4, 4, 0) AIMS_H_CASE(4, 3, 0) AIMS_H_CASE(3, 4, 0) AIMS_H_CASE(3, 3, 0)
    AIMS_H_CASE(4, 4, 1) AIMS_H_CASE(3, 3, 1)
    AIMS_H_CASE(4, 2, 0) AIMS_H_CASE(4, 1, 0) AIMS_H_CASE(3, 2, 0) AIMS_H_CASE(3, 1, 0)
    AIMS_H_CASE(2, 4, 0) AIMS_H_CASE(2, 3, 0) AIMS_H_CASE(2, 2, 0) AIMS_H_CASE(2, 1, 0)
    AIMS_H_CASE(1, 4, 0) AIMS_H_CASE(1, 3, 0) AIMS_H_CASE(1, 2, 0) AIMS_H_CASE(1, 1, 0)
    AIMS_H_CASE(2, 2, 1) AIMS_H_CASE(1, 1, 1)
    default: break;
  }
#undef AIMS_H_CASE
}

template <bool GGA>
__global__ void __launch_bounds__(kHThreads, kHCtasPerSm) k_hamiltonian(DevSys S, BatchLists L, HArgs A) {
  constexpr int NST = kHStages;
  constexpr int GW = h_group_doubles<GGA>(), SW = h_stage_doubles<GGA>();
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double *sm = reinterpret_cast<double *>(smem_raw);
  double *s_strip = sm + (size_t)NST * SW;                                  // [warps][8][kHStripLd]
  unsigned long long *s_bar = reinterpret_cast<unsigned long long *>(s_strip + kHWarps * kHStripRows * kHStripLd);   // full[NST], empty[NST]
  int *s_rowinfo = reinterpret_cast<int *>(s_bar + 2 * NST);
  int *s_colinfo = s_rowinfo + kHI;
  int *s_ld = s_colinfo + kHJ;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  __shared__ unsigned s_tix, s_warps_done;
  unsigned tix = blockIdx.x;
  if (A.det) {
    // ordered scatter: tiles are taken in list order (ascending batch) by ticket, so that every tile a CTA may have to
    // wait for below was started before it -- no deadlock whatever order the hardware dispatches CTAs in
    if (tid == 0) { s_tix = atomicAdd(A.ticket, 1u); s_warps_done = 0; }
    __syncthreads();
    tix = s_tix;
  }
  const HTile tile = A.tiles[tix];
  const int b = tile.b;
  const int nnz = L.nnz[b], nact = L.n_act[b];
  const int nnz8 = pad8(nnz), nsub = nnz8 >> 3, nblk = blk_count(nsub);
  // a stage holds 8 points (GGA: two groups, two products each) or 16 points (LDA: four groups); the LDA planes are padded
  // with zero columns to a multiple of 16 points, so that both run four product steps per barrier round trip
  constexpr int NG = h_stage_groups<GGA>();
  const int npp = round_up((int)(S.batch_ptr[b + 1] - S.batch_ptr[b]), 4 * NG);
  const int nchunk = A.pmul * (npp / (4 * NG));
  const long long boff_plane = (A.pad_off[b] - A.pad_base) * A.pmul;
  const long long fo = L.fn_off[b], ao = L.act_off[b];

  const int bI0 = tile.ti * kHIB, bI1 = min(bI0 + kHIB, nblk);
  const int bJ0 = tile.tj * kHJB, bJ1 = min(bJ0 + kHJB, nblk);
  const int rI0 = blk_start(bI0, nsub, nblk), rI1 = blk_start(bI1, nsub, nblk);
  const int rJ0 = blk_start(bJ0, nsub, nblk), rJ1 = blk_start(bJ1, nsub, nblk);

  // Live blocks (bi, bj >= bi) of this tile, enumerated column by column, are dealt to the warps in order, rotated by
  // the tile index so that the partly filled tiles along the diagonal load the four SM sub-partitions evenly.
  const int nI = bI1 - bI0, nJ = bJ1 - bJ0;
  int nlive = 0, my_bi = -1, my_bj = -1;
  const int slot = (warp + (int)(blockIdx.x & (kHWarps - 1))) & (kHWarps - 1);
  for (int cj = 0; cj < nJ; cj++) {
    const int cnt = min(nI, bJ0 + cj - bI0 + 1);                  // blocks bi = bI0 .. bI0+cnt-1 are on or above the diagonal
    if (cnt > 0) {
      if (slot >= nlive && slot < nlive + cnt) { my_bi = bI0 + slot - nlive; my_bj = bJ0 + cj; }
      nlive += cnt;
    }
  }
  const bool live = my_bi >= 0;
  const int bi = my_bi, bj = my_bj;
  int wa = 0, wb = 0, ri0 = 0, cj0 = 0;
  if (live) {
    ri0 = blk_start(bi, nsub, nblk); cj0 = blk_start(bj, nsub, nblk);
    wa = (blk_start(bi + 1, nsub, nblk) - ri0) >> 3;
    wb = (blk_start(bj + 1, nsub, nblk) - cj0) >> 3;
  }
  const bool diag = live && bi == bj;
  const int variant = live ? (wa * 4 + wb) * 2 + (diag ? 1 : 0) : -1;
  const int aoff = (ri0 - rI0) * 4 + lane, boff = (cj0 - rJ0) * 4 + lane;

  // row / column bookkeeping for the scatter
  for (int r = tid; r < kHI; r += kHThreads) s_rowinfo[r] = (rI0 + r < min(rI1, nnz)) ? L.fn_info[fo + rI0 + r] : -1;
  for (int r = tid; r < kHJ; r += kHThreads) s_colinfo[r] = (rJ0 + r < min(rJ1, nnz)) ? L.fn_info[fo + rJ0 + r] : -1;
  for (int s = tid; s < nact; s += kHThreads) s_ld[s] = L.act_ld[ao + s];

  const unsigned bar_full = smem_u32(s_bar), bar_empty = bar_full + 8 * NST;
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NST; s++) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, (unsigned)nlive); }
    mbar_fence_init();
  }
  __syncthreads();
  if (!live) return;                                              // no CTA-wide barrier below this line

  // ---- producer: chunk q -> stage q % NST; per 4-point group one contiguous segment per panel
  const double *gP = A.P + boff_plane, *gQ = A.Q + boff_plane;
  const unsigned bytesI = (unsigned)(rI1 - rI0) * 32u, bytesJ = (unsigned)(rJ1 - rJ0) * 32u;
  auto issue = [&](int q) {
    const int s = q % NST;
    const unsigned bar = bar_full + 8 * s;
    mbar_expect_tx(bar, (unsigned)NG * (GGA ? 2u : 1u) * (bytesI + bytesJ));
    const unsigned dst = smem_u32(sm + (size_t)s * SW);
#pragma unroll
    for (int g = 0; g < NG; g++) {
      const long long gI = ((long long)(NG * q + g) * nnz8 + rI0) * 4, gJ = ((long long)(NG * q + g) * nnz8 + rJ0) * 4;
      const unsigned d = dst + (unsigned)(g * GW) * 8u;
      bulk_g2s(d, gP + gI, bytesI, bar);
      bulk_g2s(d + kHI * 32u, gQ + gJ, bytesJ, bar);
      if (GGA) {
        bulk_g2s(d + (kHI + kHJ) * 32u, gQ + gI, bytesI, bar);
        bulk_g2s(d + (2 * kHI + kHJ) * 32u, gP + gJ, bytesJ, bar);
      }
    }
  };
  // the live warp in slot 0 fills the pipeline; afterwards the refill duty rotates over the live warps
  if (slot == 0 && lane == 0)
    for (int q = 0; q < min(NST, nchunk); q++) issue(q);

  double acc[4][4][2];
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int c = 0; c < 4; c++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }

  h_mma_loop<GGA>(variant, acc, sm, aoff, boff, nchunk, bar_full, bar_empty, lane, [&](int q) {
    // refill the stage released one chunk ago (lagged by one so that the wait below is normally already satisfied)
    const int qq = q - 1;
    if (qq >= 0 && qq + NST < nchunk && slot == qq % nlive) {
      mbar_wait(bar_empty + 8 * (qq % NST), (unsigned)(qq / NST) & 1u);
      issue(qq + NST);
    }
  });

  // ---- epilogue (S2d): per warp, 8-row strips through shared memory, then coalesced REDs along the block row
  if (A.det) {
    // Within one batch every H element is added to by exactly one lane of one tile, so only the order ACROSS batches
    // matters: wait until all tiles of earlier batches are done.  (`done` counts finished tiles; a tile can only finish
    // after all tiles of earlier batches, so done >= first tile of b  <=>  all earlier tiles finished.)
    const unsigned need = (unsigned)(A.tile_off[b] - A.tile_base);
    if (lane == 0) {
      unsigned seen;
      do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(seen) : "l"(A.done) : "memory"); } while (seen < need);
    }
    __syncwarp();
  }
  // AIMS_PROBE_H_EPILOGUE (probe builds only, build.py --define/--tag; results are NOT H): 0 = no scatter at all (the bound of
  // the main loop), 1 = plain stores instead of REDs (what the atomic unit costs beyond the store traffic); profiles/r02_kernel_experiments.md
#if defined(AIMS_PROBE_H_EPILOGUE) && AIMS_PROBE_H_EPILOGUE == 0
  {   // keep the accumulators live through a store that never happens (ptxas removes DMMAs whose results are dead)
    double sum = 0.0;
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
      for (int c = 0; c < 4; c++) sum += acc[a][c][0] + acc[a][c][1];
    if (sum == 12345.678) s_strip[lane] = sum;
  }
#endif
#if !defined(AIMS_PROBE_H_EPILOGUE) || AIMS_PROBE_H_EPILOGUE != 0
  double *strip = s_strip + warp * (kHStripRows * kHStripLd);
  const int fr = lane >> 2, fk = lane & 3;
  const long long *ptab = L.ptab + L.ptab_off[b];
  const int ci = (lane < wb * 8) ? s_colinfo[cj0 - rJ0 + lane] : -1;
  const int sj = ci >> 16, cb = ci & 0xFFFF;
  const int ldj = (ci >= 0) ? s_ld[sj] : 0;
  const int csub = lane >> 3;
  int cur_si = -1;                                            // atom slot of the row whose block offset is cached in `base`
  long long base = -1;
#pragma unroll
  for (int a = 0; a < 4; a++) {
    if (a < wa) {
#pragma unroll
      for (int h = 0; h < 8 / kHStripRows; h++) {
      __syncwarp();
      if (kHStripRows == 8 || (fr / kHStripRows) == h) {
#pragma unroll
        for (int c = 0; c < 4; c++)
          if (c < wb && (!diag || c >= a))
            *reinterpret_cast<double2 *>(strip + (fr % kHStripRows) * kHStripLd + c * 8 + 2 * fk) = make_double2(acc[a][c][0], acc[a][c][1]);
      }
      __syncwarp();
      if (ci >= 0 && !(diag && csub < a)) {
#pragma unroll
        for (int r = 0; r < kHStripRows; r++) {
          const int ri = s_rowinfo[ri0 - rI0 + a * 8 + h * kHStripRows + r];
          if (ri < 0) break;                                  // rows beyond nnz (zero padding) end the batch matrix
          const int si = ri >> 16, ra = ri & 0xFFFF;
          if (si > sj) continue;                              // lower atom block (only inside diagonal sub-tiles)
          if (si != cur_si) { cur_si = si; base = __ldg(ptab + si * nact + sj); }   // rows of one atom share the block
          if (base < 0) continue;                             // atom pair outside the pattern: exact zero
          const double val = strip[r * kHStripLd + lane];
#if defined(AIMS_PROBE_H_EPILOGUE) && AIMS_PROBE_H_EPILOGUE == 1
          A.H[base + (long long)ra * ldj + cb] = val;
          if (si == sj && !(diag && csub == a)) A.H[base + (long long)cb * ldj + ra] = val;
#else
          red_add_f64(A.H + base + (long long)ra * ldj + cb, val);
          // diagonal atom block holds the full square: mirror unless (col,row) is itself computed (same diagonal sub-tile)
          if (si == sj && !(diag && csub == a)) red_add_f64(A.H + base + (long long)cb * ldj + ra, val);
#endif
        }
      }
      }
    }
  }
#endif
  if (A.det) {
    __threadfence();                                   // this warp's adds are performed before it reports
    __syncwarp();
    if (lane == 0 && atomicAdd(&s_warps_done, 1u) == (unsigned)nlive - 1u) {
      __threadfence();                                 // cumulativity: the other warps' adds were fenced before their count
      atomicAdd(A.done, 1u);
    }
  }
}

}  // namespace aims
