// density.cuh -- S3a-S3d: density update n(r) = sum_ij phi_i n_ij phi_j (Eq. 3) per batch as
//   temp = D_b . Phi  (DSYMM of Fig. 6b, L359/L370)  then  n_p = sum_i Phi_ip temp_ip  (L360/L371),
//   grad n_p = 2 sum_i gradPhi_ip temp_ip  (D symmetric; L67, L93-95),
// on the FP64 tensor pipe (DMMA.8x8x4).  D_b ("calculate_density_mat", L314/L357) is never materialised: its tiles are
// gathered straight from the block-sparse D into shared memory with 8-byte cp.async.
//
// One CTA (16 warps, one per SM) per (batch, range of <= 224 points).  Warp-specialised:
//   warps 0..13  MMA warps.  The points are cut into PB <= 7 blocks of 3-4 sub-tiles of 8 points and the rows of temp
//                are walked in M-tiles of IB = min(8, 14 / PB) blocks of 3-4 sub-tiles of 8 rows; warp (pb, ib)
//                owns one 32x32-ish block, K runs over all nnz functions in stages of 16.  After an M-tile its block of
//                temp is multiplied with Phi (and grad Phi), reduced over rows with warp shuffles and added to a
//                per-(ib) partial sum in shared memory -- no atomics, deterministic.
//   warps 14,15  producers.  Per stage: the D tile (M-tile rows x 16 functions) by 8-byte cp.async gathers, and the Phi
//                rows of the stage for all points by ONE bulk async copy (contiguous in the density layout).
// Stages are handed over with mbarriers (full: producer -> MMA, empty: MMA -> producer); there is no CTA-wide barrier
// in the main loop, and every DMMA is unpredicated straight-line code (see hamiltonian.cuh for the measurements).
#pragma once
#include "common.cuh"
#include "hamiltonian.cuh"   // blk_start / blk_count

namespace aims {

#ifndef AIMS_D_NP
#define AIMS_D_NP 224
#endif
#ifndef AIMS_D_STAGES
#define AIMS_D_STAGES 4
#endif
constexpr int kDKC = 16;            // K (functions j) per stage
constexpr int kDNP = AIMS_D_NP;     // max points per CTA (7 blocks of 32)
constexpr int kDStages = AIMS_D_STAGES;
constexpr int kDThreads = 512;
constexpr int kDMmaWarps = 14;             // MMA warps of a CTA with 5..7 point blocks (129..224 points)
constexpr int kDProdLanes = 64;            // ... and its producer lanes (2 warps)
// CTAs with <= 4 point blocks (<= 128 points) run 12 MMA warps and FOUR producer warps: the D_b tile of a stage has the
// same number of rows per DMMA whatever the point count, so a short batch needs 2-3x more gather per flop, and round 1
// measured its two producer warps as the limiter (17.6 TFLOP/s at 64-point batches); 12 warps, three per SM
// sub-partition, still saturate the FP64 pipe (profiles/r01_dmma_probe.md: 8 warps reach 99.7 %).
__host__ __device__ inline int d_mma_warps(int PB) { return PB <= 4 ? 12 : 14; }
// One pipeline stage holds the D tile (M-tile rows x 16) followed by the Phi tile (CTA points x 16).  With PB point
// blocks and IB = min(4, 14 / PB) row blocks per M-tile, rows + points never exceed 64 + 224 (PB = 7, IB = 2).
constexpr int kDStageRows = 64 + kDNP;             // rows of D plus points of Phi per stage
constexpr int kDStage = kDStageRows * kDKC;        // doubles per stage
constexpr int kDPartCols = 448;                    // max of (row blocks per M-tile) x (points of the CTA): 7 x 64
constexpr int kDPrefetchLead = 6;                  // stages before the M-tile epilogue at which its operands are prefetched to L2

// AIMS_PROBE_WARP_CYCLES (probe builds only): per-warp cycle counters -- [0] waiting for a stage (MMA warps: full barrier,
// producers: empty barrier), [1] M-tile epilogues (MMA warps) / gather + copy issue (producers); a few CTAs print theirs.
#ifdef AIMS_PROBE_WARP_CYCLES
__device__ __forceinline__ long long *probe_wc() { __shared__ long long s[20][4]; return s[threadIdx.x >> 5]; }
#define AIMS_TIMED(idx, ...) { const long long t0_ = clock64(); __VA_ARGS__; if ((threadIdx.x & 31) == 0) probe_wc()[idx] += clock64() - t0_; }
#else
#define AIMS_TIMED(idx, ...) { __VA_ARGS__; }
#endif

#ifdef AIMS_PROBE_D_NO_HANDSHAKE
#define AIMS_HS(...)
#else
#define AIMS_HS(...) __VA_ARGS__
#endif

struct DItem { int b, p0, npt, pad; };     // points [p0, p0+npt) of batch b; p0 and npt multiples of 8

struct DArgs {
  const DItem *items;
  const int *order;                 // launch order: CTA x works on items[order[x]] (NULL: items[x])
  const double *P;                  // Phi plane
  const double *G[3];               // gradient planes (GRAD only)
  const long long *pad_off;         // [n_batches+1] prefix of round_up(nnz,16)*pad8(np) (density layout)
  long long pad_base;
  const double *D;                  // block-sparse density matrix
  double *n, *gn;                   // outputs [n_points], [3][n_points]
  long long n_points;
  int max_nnz_pad;                  // capacity of the fn_info smem array
  int ptab_in_smem;                 // the batch's atom-pair offset table is staged in shared memory
};

inline size_t d_smem_bytes(int max_nnz, int max_act, bool ptab_in_smem) {
  size_t s = (size_t)kDStages * kDStage * sizeof(double);
  s += (size_t)4 * kDPartCols * sizeof(double);               // part[ib][q][col of the CTA], IB * npt <= kDPartCols
  s += 2 * kDStages * sizeof(unsigned long long);             // full / empty barriers
  if (ptab_in_smem) s += (size_t)max_act * max_act * sizeof(long long);
  s += (size_t)pad8(max_nnz) * sizeof(int) + (size_t)kMaxActive * sizeof(int);
  return s;
}

// The K loop of one warp block of (8 WA rows) x (8 WB points) over nkc pipeline stages, as ONE instruction stream.
// Operand fragments are reloaded from shared memory in place WHILE the DMMAs of the current step are issued -- an A
// fragment is dead once its row of DMMAs is issued, a B fragment once the last row has used it -- and the reloads of a
// stage's last step already fetch the first step of the NEXT stage (its "full" barrier is waited for after the first
// row of DMMAs is in the pipe).  So the warp's DMMA issue never pauses for a load, a barrier round trip or loop control
// between the first and the last stage.  Why it matters: the warps of an SM sub-partition share its FP64 pipe
// round-robin and therefore reach every stage boundary together, so per-stage bubbles of the individual warps do NOT
// overlap with each other's DMMAs (measured per-warp cycle counters: boundary work was 6.5 % of the run time).
// Micro-benchmark on the B200 (8 LDS.64 + 16 DMMA per step): one warp per sub-partition reaches 79 % of the pipe peak
// with load-then-compute steps and 92 % with overlapped loads; four warps 94 % -> 99.6 %.
// step: running stage counter of the CTA (stage = step % kDStages, parity from step / kDStages), advanced by nkc.
// --define AIMS_D_UNROLL_STAGE=1 (probe builds): the K loop below with the four steps of a full stage as ONE straight-line block.
#ifndef AIMS_D_UNROLL_STAGE
#define AIMS_D_UNROLL_STAGE 0
#endif
#if AIMS_D_UNROLL_STAGE
// One K step of a (WA x WB) block: DMMAs row by row, every fragment reloaded in place from (a1, b1) as soon as it is dead.
// LAST (compile time): the last step of a stage -- after the first row of DMMAs is in the pipe, make sure the next stage has
// landed and redirect the reloads to it.
template <int WA, int WB, bool LAST>
__device__ __forceinline__ void d_step(double (&acc)[4][4][2], double (&fa)[WA], double (&fb)[WB], const double *a1, const double *b1,
                                       const double *&tA, const double *&tB, const double *sAl, const double *sBl, bool more_stages,
                                       int step, unsigned bar_full) {
#pragma unroll
  for (int c = 0; c < WB; c++) dmma8x8x4(acc[0][c][0], acc[0][c][1], fa[0], fb[c]);
  if (LAST) {
    if (more_stages) {
      const int s1 = (step + 1) % kDStages;
      AIMS_HS(AIMS_TIMED(0, mbar_wait(bar_full + 8 * s1, (unsigned)((step + 1) / kDStages) & 1u)))
      a1 = sAl + (size_t)s1 * kDStage; b1 = sBl + (size_t)s1 * kDStage;
    } else {
      a1 = tA; b1 = tB;                      // nothing follows: harmless reload of this stage's first step
    }
  }
  if (WA > 1) {
    fa[0] = a1[0];
#pragma unroll
    for (int a = 1; a < WA - 1; a++) {
#pragma unroll
      for (int c = 0; c < WB; c++) dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
      fa[a] = a1[a * 32];
    }
#pragma unroll
    for (int c = 0; c < WB; c++) {
      dmma8x8x4(acc[WA - 1][c][0], acc[WA - 1][c][1], fa[WA - 1], fb[c]);
      fb[c] = b1[c * (2 * kDKC * 4)];
    }
    fa[WA - 1] = a1[(WA - 1) * 32];
  } else {
    fa[0] = a1[0];
#pragma unroll
    for (int c = 0; c < WB; c++) fb[c] = b1[c * (2 * kDKC * 4)];
  }
  if (LAST) { tA = a1; tB = b1; }
}

// nnz(B) and the stage count come from global memory, so the compiler cannot prove the loop counters warp-uniform and guards
// the DMMAs of every basic block with a WARPSYNC after a predicated branch.  aims_gpu_dmma_probe variants 5 / 10 / 11
// (profiles/r02_dmma_probe.md): the same K step reaches 99.7 % of the pipe in a uniform loop, 96.2 % inside this control flow
// with one step per iteration, 98.5 % with the four steps of a stage unrolled (four warps per pipe; 98 / 90 / 95.5 % with two).
// In the kernels the unrolled form (--define AIMS_D_UNROLL_STAGE=1) is a wash: k_density 388.2 instead of 392.2 ms on config 5,
// but 117.6 instead of 115.1 ms on 64-point batches and 10.50 instead of 10.40 ms on config 3 (profiles/r02_kernel_experiments.md).
template <int WA, int WB>
__device__ __forceinline__ void d_mma_kloop_t(double (&acc)[4][4][2], const double *sAl, const double *sBl, int tm, int nkc,
                                              int nnz8, int &step, unsigned bar_full, unsigned bar_empty, int lane) {
  int s = step % kDStages;
  AIMS_HS(AIMS_TIMED(0, mbar_wait(bar_full + 8 * s, (unsigned)(step / kDStages) & 1u)))
  const double *tA = sAl + (size_t)s * kDStage, *tB = sBl + (size_t)s * kDStage;
  const int tm4 = tm * 4;
  double fa[WA], fb[WB];
#pragma unroll
  for (int a = 0; a < WA; a++) fa[a] = tA[a * 32];
#pragma unroll
  for (int c = 0; c < WB; c++) fb[c] = tB[c * (2 * kDKC * 4)];
#pragma unroll 1
  for (int kc = 0; kc < nkc; kc++) {
    const int nk4 = min(kDKC, nnz8 - kc * kDKC) >> 2;
    const bool more_stages = kc + 1 < nkc;
    if (nk4 == 4) {
      d_step<WA, WB, false>(acc, fa, fb, tA + tm4, tB + 16, tA, tB, sAl, sBl, more_stages, step, bar_full);
      d_step<WA, WB, false>(acc, fa, fb, tA + 2 * tm4, tB + 32, tA, tB, sAl, sBl, more_stages, step, bar_full);
      d_step<WA, WB, false>(acc, fa, fb, tA + 3 * tm4, tB + 48, tA, tB, sAl, sBl, more_stages, step, bar_full);
      d_step<WA, WB, true>(acc, fa, fb, tA, tB, tA, tB, sAl, sBl, more_stages, step, bar_full);
    } else {
#pragma unroll 1
      for (int t = 0; t < nk4; t++) {
        if (t + 1 == nk4) d_step<WA, WB, true>(acc, fa, fb, tA, tB, tA, tB, sAl, sBl, more_stages, step, bar_full);
        else d_step<WA, WB, false>(acc, fa, fb, tA + (t + 1) * tm4, tB + (t + 1) * 16, tA, tB, sAl, sBl, more_stages, step, bar_full);
      }
    }
    // every fragment of stage s is in registers (the reloads above already read the next stage): release it
    __syncwarp();
    AIMS_HS(if (lane == 0) mbar_arrive(bar_empty + 8 * s);)
    step++;
    s = step % kDStages;
  }
}

#else
template <int WA, int WB>
__device__ __forceinline__ void d_mma_kloop_t(double (&acc)[4][4][2], const double *sAl, const double *sBl, int tm, int nkc,
                                              int nnz8, int &step, unsigned bar_full, unsigned bar_empty, int lane) {
  int s = step % kDStages;
  AIMS_HS(AIMS_TIMED(0, mbar_wait(bar_full + 8 * s, (unsigned)(step / kDStages) & 1u)))
  const double *tA = sAl + (size_t)s * kDStage, *tB = sBl + (size_t)s * kDStage;
  double fa[WA], fb[WB];
#pragma unroll
  for (int a = 0; a < WA; a++) fa[a] = tA[a * 32];
#pragma unroll
  for (int c = 0; c < WB; c++) fb[c] = tB[c * (2 * kDKC * 4)];
#pragma unroll 1
  for (int kc = 0; kc < nkc; kc++) {
    const int nk4 = min(kDKC, nnz8 - kc * kDKC) >> 2;
    const bool more_stages = kc + 1 < nkc;
#pragma unroll 1
    for (int t = 0; t < nk4; t++) {
      const bool last = t + 1 == nk4;
      const double *a1 = tA + (t + 1) * tm * 4, *b1 = tB + (t + 1) * 16;
      // first row of DMMAs, then (last step of the stage) make sure the next stage has landed before reloading from it
#pragma unroll
      for (int c = 0; c < WB; c++) dmma8x8x4(acc[0][c][0], acc[0][c][1], fa[0], fb[c]);
      if (last) {
        if (more_stages) {
          const int s1 = (step + 1) % kDStages;
          AIMS_HS(AIMS_TIMED(0, mbar_wait(bar_full + 8 * s1, (unsigned)((step + 1) / kDStages) & 1u)))
          a1 = sAl + (size_t)s1 * kDStage; b1 = sBl + (size_t)s1 * kDStage;
        } else {
          a1 = tA; b1 = tB;                      // nothing follows: harmless reload of this stage's first step
        }
      }
      if (WA > 1) {
        fa[0] = a1[0];
#pragma unroll
        for (int a = 1; a < WA - 1; a++) {
#pragma unroll
          for (int c = 0; c < WB; c++) dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
          fa[a] = a1[a * 32];
        }
#pragma unroll
        for (int c = 0; c < WB; c++) {
          dmma8x8x4(acc[WA - 1][c][0], acc[WA - 1][c][1], fa[WA - 1], fb[c]);
          fb[c] = b1[c * (2 * kDKC * 4)];
        }
        fa[WA - 1] = a1[(WA - 1) * 32];
      } else {
        fa[0] = a1[0];
#pragma unroll
        for (int c = 0; c < WB; c++) fb[c] = b1[c * (2 * kDKC * 4)];
      }
      if (last) { tA = a1; tB = b1; }
    }
    // every fragment of stage s is in registers (the reloads above already read the next stage): release it
    __syncwarp();
    AIMS_HS(if (lane == 0) mbar_arrive(bar_empty + 8 * s);)
    step++;
    s = step % kDStages;
  }
}

#endif

// K loop of a warp without a block in this M-tile: it only takes part in the stage hand-over
__device__ __forceinline__ void d_idle_kloop(int nkc, int &step, unsigned bar_full, unsigned bar_empty, int lane) {
#pragma unroll 1
  for (int kc = 0; kc < nkc; kc++, step++) {
    const int s = step % kDStages;
    AIMS_HS(mbar_wait(bar_full + 8 * s, (unsigned)(step / kDStages) & 1u);)
    __syncwarp();
    AIMS_HS(if (lane == 0) mbar_arrive(bar_empty + 8 * s);)
  }
}

__device__ __forceinline__ void d_mma_kloop(int variant, double (&acc)[4][4][2], const double *sAl, const double *sBl, int tm,
                                            int nkc, int nnz8, int &step, unsigned bar_full, unsigned bar_empty, int lane) {
#define AIMS_D_CASE(WA, WB)                                                                               \
  case WA * 4 + WB:                                                                                       \
    d_mma_kloop_t<WA, WB>(acc, sAl, sBl, tm, nkc, nnz8, step, bar_full, bar_empty, lane);                 \
    break;
  switch (variant) {
    AIMS_D_CASE(4, 4) AIMS_D_CASE(4, 3) AIMS_D_CASE(3, 4) AIMS_D_CASE(3, 3)
    AIMS_D_CASE(4, 2) AIMS_D_CASE(4, 1) AIMS_D_CASE(3, 2) AIMS_D_CASE(3, 1)
    AIMS_D_CASE(2, 4) AIMS_D_CASE(2, 3) AIMS_D_CASE(2, 2) AIMS_D_CASE(2, 1)
    AIMS_D_CASE(1, 4) AIMS_D_CASE(1, 3) AIMS_D_CASE(1, 2) AIMS_D_CASE(1, 1)
    default: d_idle_kloop(nkc, step, bar_full, bar_empty, lane); break;
  }
#undef AIMS_D_CASE
}

// Producer side of one K stage: the tile D_b[i0 + r][k0 .. k0+15], r < tm, of the symmetric block-sparse matrix M restricted
// to nnz(B) ("calculate_density_mat"), written as [4-function group][row][4] into dA.  pl = 0..63.
__device__ __forceinline__ void d_gather_tile(double *dA, const double *M, int i0, int tm, int k0, int nnz, int nnz8, int nact,
                                              const int *sInfo, const int *sLd, const long long *ptab, int pl, int nprod) {
  // D_b[i0 + r][k0 + 4t .. +3]: one (row, 4-function group) unit = four 8-byte copies, gathered from the block pattern
  // (stored block (si,sj) for si <= sj, transposed read of block (sj,si) below the diagonal).  The column side of a stage is
  // the same for every row, so it is decoded once per lane (registers); a row is decoded once per stage; what is left per
  // unit is one table look-up (block offset of the atom pair) and the address -- four independent units per row.
  const int ng = min(kDKC, nnz8 - k0) >> 2;          // 4-function groups with at least one real function
  int sjt[4], cjt[4], ldjt[4];                       // atom slot / first column / ld of group t; sjt < 0: not 4 functions of one atom
#pragma unroll
  for (int t = 0; t < 4; t++) {
    sjt[t] = -1; cjt[t] = 0; ldjt[t] = 0;
    if (t < ng) {
      const int4 fj4 = *reinterpret_cast<const int4 *>(sInfo + k0 + 4 * t);   // sInfo is padded with -1 up to nnz8
      if (fj4.w >= 0 && (fj4.x >> 16) == (fj4.w >> 16) && (fj4.w - fj4.x) == 3) {
        sjt[t] = fj4.x >> 16; cjt[t] = fj4.x & 0xFFFF; ldjt[t] = sLd[sjt[t]];
      }
    }
  }
  for (int r = pl; r < tm; r += nprod) {             // consecutive lanes -> consecutive rows (transposed reads coalesce)
    const int i = i0 + r;
    if (i >= nnz) {
#pragma unroll
      for (int t = 0; t < 4; t++)
        if (t < ng) {
          const unsigned dst = smem_u32(dA + (t * tm + r) * 4);
#pragma unroll
          for (int q = 0; q < 4; q++) cp_async8(dst + 8u * q, M, 0);
        }
      continue;
    }
    const int fi = sInfo[i];
    const int si = fi >> 16, ri = fi & 0xFFFF;
    const long long *prow = ptab + si * nact;
    const int ldi = sLd[si];
#pragma unroll
    for (int t = 0; t < 4; t++) {
      if (t >= ng) continue;
      const unsigned dst = smem_u32(dA + (t * tm + r) * 4);
      if (sjt[t] >= 0) {
        // fast path: four consecutive functions of one atom
        const int sj = sjt[t];
        const long long base = prow[sj];
        const double *src = M;
        long long stride = 0;
        int bytes = 0;
        if (base >= 0) {
          bytes = 8;
          if (si <= sj) { src = M + base + (long long)ri * ldjt[t] + cjt[t]; stride = 1; }
          else { src = M + base + (long long)cjt[t] * ldi + ri; stride = ldi; }
        }
#pragma unroll
        for (int q = 0; q < 4; q++) cp_async8(dst + 8u * q, src + q * stride, bytes);
      } else {
#pragma unroll
        for (int q = 0; q < 4; q++) {
          const int fj = sInfo[k0 + 4 * t + q];
          const double *src = M;
          int bytes = 0;
          if (fj >= 0) {
            const int sj = fj >> 16, cj = fj & 0xFFFF;
            const long long base = prow[sj];
            if (base >= 0) {
              src = (si <= sj) ? M + base + (long long)ri * sLd[sj] + cj : M + base + (long long)cj * ldi + ri;
              bytes = 8;
            }
          }
          cp_async8(dst + 8u * q, src, bytes);
        }
      }
    }
  }
}

// Deal the PB*IB blocks (work ~ point sub-tiles wb) to the MMA warps so that the four SM sub-partitions carry equal
// DMMA load: sub-partition q hosts MMA warps q, q+4, q+8(, q+12) -- 2 and 3 have only three because the producers
// sit there.  Blocks in descending size go to the sub-partition whose remaining slots need the largest average.
// s_map[warp] = pb | ib << 8, -1 = idle.  One thread.
__device__ __forceinline__ void d_deal_blocks(int *s_map, int PB, int IB, int psub, int nmma = kDMmaWarps) {
  const int nb = PB * IB;
  int cnt[4], load[4] = {0, 0, 0, 0}, used[4] = {0, 0, 0, 0}, total = 0;
  for (int q = 0; q < 4; q++) cnt[q] = nb / 4 + (q < (nb & 3) ? 1 : 0);
  for (int w = 0; w < nmma; w++) s_map[w] = -1;
  for (int pb2 = 0; pb2 < PB; pb2++) total += IB * ((blk_start(pb2 + 1, psub, PB) - blk_start(pb2, psub, PB)) >> 3);
  for (int sz = 4; sz >= 1; sz--)
    for (int pb2 = 0; pb2 < PB; pb2++) {
      if (((blk_start(pb2 + 1, psub, PB) - blk_start(pb2, psub, PB)) >> 3) != sz) continue;
      for (int ib2 = 0; ib2 < IB; ib2++) {
        int best = -1;
        for (int q = 0; q < 4; q++) {
          if (used[q] >= cnt[q]) continue;
          if (best < 0 || (total - 4 * load[q]) * (cnt[best] - used[best]) > (total - 4 * load[best]) * (cnt[q] - used[q])) best = q;
        }
        s_map[best + 4 * used[best]] = pb2 | (ib2 << 8);
        used[best]++; load[best] += sz;
      }
    }
}

// NMMA: 14 or 12 MMA warps (d_mma_warps); a compile-time constant inside the body, selected per CTA by the kernel below.
template <bool GRAD, int NMMA>
__device__ __forceinline__ void d_density_body(const DevSys &S, const BatchLists &L, const DArgs &A, int max_act, const DItem it) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double *sA = reinterpret_cast<double *>(smem_raw);                     // stage s: [k4][tm][4] at sA + s * kDStage
  double *sPart = sA + (size_t)kDStages * kDStage;                       // [ib][q][col]
  unsigned long long *s_bar = reinterpret_cast<unsigned long long *>(sPart + 4 * kDPartCols);
  int *sInfo = reinterpret_cast<int *>(s_bar + 2 * kDStages);           // 16-byte aligned; [pad8(max nnz)]
  int *sLd = sInfo + pad8(A.max_nnz_pad);
  long long *sPtab = reinterpret_cast<long long *>(sLd + kMaxActive);

  const int b = it.b;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nnz = L.nnz[b], nact = L.n_act[b];
  const int nnz8 = pad8(nnz), nsub = nnz8 >> 3, nblk = blk_count(nsub);
  const long long pbase = S.batch_ptr[b];
  const int np = (int)(S.batch_ptr[b + 1] - pbase);
  const long long boff = A.pad_off[b] - A.pad_base;
  const int p0 = it.p0, npt = it.npt;                    // this CTA's points [p0, p0+npt) of the batch (multiples of 8)
  const int psub = npt >> 3, PB = blk_count(psub);       // point sub-tiles and blocks
  constexpr int nmma = NMMA, nprod = (16 - NMMA) * 32;         // MMA warps and producer lanes of this CTA
  const int IB = min(8, nmma / PB);                // row blocks per M-tile: 2,2,2,3,4,7,8 for PB = 7..1
  const int n_mt = (nblk + IB - 1) / IB;                 // M-tiles
  const double *sB = sA + IB * 32 * kDKC;                // stage s: [point group][16][4] at sB + s * kDStage
  const int nkc = (nnz8 + kDKC - 1) / kDKC;              // K stages per M-tile
  const long long fo = L.fn_off[b], ao = L.act_off[b];
  const long long *gptab = L.ptab + L.ptab_off[b];

  for (int i = tid; i < nnz8; i += kDThreads) sInfo[i] = i < nnz ? L.fn_info[fo + i] : -1;
  for (int i = tid; i < nact; i += kDThreads) sLd[i] = L.act_ld[ao + i];
  if (A.ptab_in_smem)
    for (int i = tid; i < nact * nact; i += kDThreads) sPtab[i] = gptab[i];
  for (int i = tid; i < 4 * kDPartCols; i += kDThreads) sPart[i] = 0.0;
  const unsigned bar_full = smem_u32(s_bar), bar_empty = bar_full + 8 * kDStages;
  __shared__ int s_map[kDMmaWarps];                      // MMA warp -> (pb | ib << 8), -1 = idle
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kDStages; s++) {
      mbar_init(bar_full + 8 * s, (unsigned)nprod + 1u);  // the producers' cp.async completions + the expect_tx arrival
      mbar_init(bar_empty + 8 * s, (unsigned)nmma);
    }
    mbar_fence_init();
    d_deal_blocks(s_map, PB, IB, psub, nmma);
  }
  __syncthreads();
#ifdef AIMS_PROBE_WARP_CYCLES
  if (lane == 0) { long long *w = probe_wc(); w[0] = 0; w[1] = 0; w[2] = clock64(); }
  __syncwarp();
#endif
  const long long *ptab = A.ptab_in_smem ? sPtab : gptab;
  const double *gP = A.P + boff;

  if (warp >= nmma) {
    // =========================================================================== producers
#ifdef AIMS_PROBE_D_NO_HANDSHAKE
    if (warp >= nmma) return;
#endif
    const int pl = tid - nmma * 32;                // 0..63
    const int np8 = pad8(np);
    int step = 0;
#pragma unroll 1
    for (int mt = 0; mt < n_mt; mt++) {
      const int bi0 = mt * IB, bi1 = min(bi0 + IB, nblk);
      const int i0 = blk_start(bi0, nsub, nblk), tm = blk_start(bi1, nsub, nblk) - i0;
#pragma unroll 1
      for (int kc = 0; kc < nkc; kc++, step++) {
      const int s = step % kDStages;
      if (step >= kDStages) AIMS_TIMED(0, mbar_wait(bar_empty + 8 * s, (unsigned)(step / kDStages - 1) & 1u))
      const int k0 = kc * kDKC;
#ifdef AIMS_PROBE_WARP_CYCLES
      const long long tg0 = clock64();
#endif
      if (kc == max(nkc - kDPrefetchLead, 0)) {
        // operands of this M-tile's epilogue (rows [i0, i0+tm) of Phi and grad Phi at the CTA's points): whole 16-row
        // chunks are contiguous in the density layout -> one bulk L2 prefetch per chunk and plane
        const int c0 = i0 >> 4, nch = ((i0 + tm - 1) >> 4) - c0 + 1;
        for (int idx = pl; idx < nch * (GRAD ? 4 : 1); idx += nprod) {
          const int c = c0 + (GRAD ? (idx >> 2) : idx), q = GRAD ? (idx & 3) : 0;
          const double *base = (q == 0) ? gP : A.G[q - 1] + boff;
          bulk_prefetch_l2(base + ((long long)c * (np8 >> 2) + (p0 >> 2)) * 64, (unsigned)npt * 128u);
        }
      }
      // AIMS_PROBE_D_NO_BULK / _NO_GATHER / _NO_HANDSHAKE (probe builds only; results are NOT n): what each part of the
      // producer -> MMA hand-over costs, profiles/r02_kernel_experiments.md
      if (pl == nprod - 1) {
        // Phi rows [k0, k0+16) of every point of the CTA: ONE contiguous segment in the density layout
#ifdef AIMS_PROBE_D_NO_BULK
        mbar_arrive(bar_full + 8 * s);
#else
        mbar_expect_tx(bar_full + 8 * s, (unsigned)npt * 128u);
        bulk_g2s(smem_u32(sB + (size_t)s * kDStage), gP + ((long long)kc * (np8 >> 2) + (p0 >> 2)) * 64, (unsigned)npt * 128u,
                 bar_full + 8 * s);
#endif
      }
#ifndef AIMS_PROBE_D_NO_GATHER
      d_gather_tile(sA + (size_t)s * kDStage, A.D, i0, tm, k0, nnz, nnz8, nact, sInfo, sLd, ptab, pl, nprod);
#endif
      cp_async_mbar_arrive_noinc(bar_full + 8 * s);
#ifdef AIMS_PROBE_WARP_CYCLES
      if (lane == 0) probe_wc()[1] += clock64() - tg0;
#endif
      }
    }
  } else {
    // =========================================================================== MMA warps
    const int wmap = s_map[warp];
    const bool wlive = wmap >= 0;
    const int pb = wmap & 0xFF, ib = wlive ? (wmap >> 8) : 0;
    const int ps0 = wlive ? blk_start(pb, psub, PB) : 0;                       // first point (within the CTA) of my block
    const int wb = wlive ? (blk_start(pb + 1, psub, PB) - ps0) >> 3 : 0;
    const int fr = lane >> 2, fk = lane & 3;
    const int np8 = pad8(np);
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
      d_mma_kloop(blive ? variant : 0, acc, sA + aoffl, sB + boffl, tm, nkc, nnz8, step, bar_full, bar_empty, lane);

#ifdef AIMS_PROBE_WARP_CYCLES
      const long long te0 = clock64();
#endif
      // AIMS_PROBE_NO_D_EPILOGUE (probe builds only; results are NOT n): the bound of the K loops alone; the accumulators stay
      // live through a store that never happens (ptxas removes DMMAs whose results are dead)
#ifdef AIMS_PROBE_NO_D_EPILOGUE
      if (blive) {
        double sum = 0.0;
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
          for (int c = 0; c < 4; c++) sum += acc[a][c][0] + acc[a][c][1];
        if (sum == 12345.678) sPart[lane] = sum;
      }
      if (false) {
#else
      if (blive) {
#endif
        // ---- M-tile epilogue: n_p += sum_i Phi_ip temp_ip (and gradient), rows reduced by shuffles
#pragma unroll
        for (int c = 0; c < 4; c++) {
          if (c < wb) {
            const int col = ps0 + c * 8 + 2 * fk;            // within the CTA's point range (even)
            const int p = p0 + col;                          // within the batch
            double sn[2] = {0.0, 0.0}, sg[3][2] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
            // two row sub-tiles at a time: all their loads (L2-prefetched by the producers) are issued before the first
            // FMA, so that an epilogue costs 2 x wb load round trips instead of 4 x wb
            constexpr int NQ = GRAD ? 4 : 1;
#pragma unroll
            for (int a0 = 0; a0 < 4; a0 += 2) {
              if (a0 < wa) {
                double2 ev[2][NQ];
#pragma unroll
                for (int da = 0; da < 2; da++) {
                  const int i = ri0 + min(a0 + da, wa - 1) * 8 + fr;   // < nnz8: padding rows are zero in the planes
                  const long long o = (((long long)(i >> 4) * (np8 >> 2) + (p >> 2)) * 16 + (i & 15)) * 4 + (p & 3);
                  ev[da][0] = __ldg(reinterpret_cast<const double2 *>(gP + o));
                  if (GRAD)
#pragma unroll
                    for (int q = 0; q < 3; q++) ev[da][q + 1] = __ldg(reinterpret_cast<const double2 *>(A.G[q] + boff + o));
                }
#pragma unroll
                for (int da = 0; da < 2; da++) {
                  if (a0 + da < wa) {
                    sn[0] += ev[da][0].x * acc[a0 + da][c][0];
                    sn[1] += ev[da][0].y * acc[a0 + da][c][1];
                    if (GRAD)
#pragma unroll
                      for (int q = 0; q < 3; q++) {
                        sg[q][0] += ev[da][q + 1].x * acc[a0 + da][c][0];
                        sg[q][1] += ev[da][q + 1].y * acc[a0 + da][c][1];
                      }
                  }
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
            if (fr == 0) {   // lanes 0..3 own columns 2*fk, 2*fk+1; (ib, column) has exactly one owner warp -> no race
              double *pp = sPart + (ib * 4) * npt + col;
              pp[0] += sn[0]; pp[1] += sn[1];
              if (GRAD)
#pragma unroll
                for (int q = 0; q < 3; q++) { pp[(q + 1) * npt] += sg[q][0]; pp[(q + 1) * npt + 1] += sg[q][1]; }
            }
          }
        }
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
          for (int c = 0; c < 4; c++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }
      }
#ifdef AIMS_PROBE_WARP_CYCLES
      if (lane == 0) probe_wc()[1] += clock64() - te0;
#endif
    }
  }
  __syncthreads();
#ifdef AIMS_PROBE_WARP_CYCLES
  if ((blockIdx.x & 1023) == 517 && lane == 0) {
    const long long *w = probe_wc();
    printf("WC cta %d b %d nnz %d npt %d warp %2d %s map %d total %lld wait %lld %s %lld\n", (int)blockIdx.x, b, nnz, npt, warp,
           warp >= nmma ? "prod" : "mma ", warp < nmma ? s_map[warp] : -1, clock64() - w[2], w[0], warp >= nmma ? "gather" : "epilogue", w[1]);
  }
#endif

  // ---- S3d: store (mapping to the global point array is the identity on the batch's contiguous range)
  for (int col = tid; col < npt; col += kDThreads) {
    const int p = p0 + col;
    if (p >= np) continue;
    double v = 0.0;
    for (int m = 0; m < IB; m++) v += sPart[(m * 4) * npt + col];
    A.n[pbase + p] = v;
    if (GRAD)
#pragma unroll
      for (int q = 0; q < 3; q++) {
        double u = 0.0;
        for (int m = 0; m < IB; m++) u += sPart[(m * 4 + q + 1) * npt + col];
        A.gn[(long long)q * A.n_points + pbase + p] = 2.0 * u;
      }
  }
}

template <bool GRAD>
__global__ void __launch_bounds__(kDThreads, 1) k_density(DevSys S, BatchLists L, DArgs A, int max_act) {
  const DItem it = A.items[A.order ? A.order[blockIdx.x] : blockIdx.x];
  if (d_mma_warps(blk_count(it.npt >> 3)) == 12) d_density_body<GRAD, 12>(S, L, A, max_act, it);
  else d_density_body<GRAD, 14>(S, L, A, max_act, it);
}

}  // namespace aims
