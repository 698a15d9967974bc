// density_b.cuh -- MEASURED AND REJECTED VARIANT of density.cuh (probe builds only: --define AIMS_PROBE_BALANCED_DENSITY=1;
// numbers in profiles/r02_kernel_experiments.md, section 3).  S3a-S3d for CTAs of 192 or 200 points with EQUAL DMMA work for
// every MMA warp and every SM sub-partition.
//
// The question it answers.  k_density has 14 MMA warps of 12 or 16 DMMAs per K step, 52/52/48/48 per sub-partition (three warps
// hold at most 3 x 16 accumulator sub-tiles; 96.2 % bound), and its lighter warps wait 10-17 % of their time at the stage ring.
// Is that imbalance what keeps the kernel at 80 % of the FP64 pipe?  Here: 18 warps.  Warps 0..15 are MMA warps: row block ib (the
// M-tile's <= 8 row sub-tiles are cut in two blocks of <= 4) x column group pb (3 point sub-tiles, points [24 pb, 24 pb + 24)) --
// a 4 x 3 block, 12 DMMAs per K step; every sub-partition hosts two warps of either row block.  A 200-point CTA has a 25th
// point sub-tile (8 more DMMAs per step): its piece (ib, h) -- rows 2h, 2h+1 of row block ib -- is shared by the four warps
// (pb = 2 qx + h, ib), qx = 0..3, which take turns over the four K steps of a stage and each keep a partial accumulator
// (summed in the epilogue's shared-memory slots).  Every warp issues exactly 4 x 12 + 2 = 50 DMMAs per stage.  Warps 16, 17 are
// the producers, as in density.cuh.  576 threads leave 112 registers per thread; the 4 x 3 (+2) accumulators need 56.
// Answer: parity green, 406.5 ms against 392.2 ms on config 5 -- balance is NOT the limiter; density.cuh stays the product.
#pragma once
#include "density.cuh"

namespace aims {

constexpr int kBThreads = 576;
constexpr int kBMma = 16;                  // MMA warps
constexpr int kBProd = 64;                 // producer lanes
constexpr int kBSlots = 2;                 // partial-sum slots per column of the 4 x 3 blocks: ib
constexpr int kBXSlots = 16;               // ... and of the 25th point sub-tile: (ib, h, qx)
constexpr int kBMinSub = 24, kBMaxSub = 25;   // point sub-tiles of an item this kernel takes

__host__ __device__ inline bool b_item_ok(int npt) { return (npt >> 3) >= kBMinSub && (npt >> 3) <= kBMaxSub; }

inline size_t b_smem_bytes(int max_nnz, int max_act, bool ptab_in_smem) {
  size_t s = (size_t)kDStages * kDStage * sizeof(double);
  s += (size_t)(kBSlots * 4 * 8 * kBMinSub + kBXSlots * 4 * 8) * sizeof(double);   // part[ib][q][192], partx[slot][q][8]
  s += 2 * kDStages * sizeof(unsigned long long);
  if (ptab_in_smem) s += (size_t)max_act * max_act * sizeof(long long);
  s += (size_t)pad8(max_nnz) * sizeof(int) + (size_t)kMaxActive * sizeof(int);
  return s;
}

// K loop of one MMA warp over nkc stages: a (WA x 3) block, plus -- in K step tx of every stage -- XN <= 2 extra DMMAs on rows
// X0 .. X0+XN-1 of the block and the CTA's 25th point sub-tile.  Same instruction-stream discipline as d_mma_kloop_t
// (density.cuh): fragments are reloaded in place while the step's DMMAs issue (an A fragment is dead after its row, a B
// fragment after the last row), the last step of a stage already loads from the next one, whose "full" barrier is waited
// for after the first row of DMMAs is in the pipe; the extra B fragment is fetched once per stage.
// One K step.  XS: this step also carries the warp's piece of the 25th point sub-tile.  A compile-time flag on purpose: a
// DMMA that is merely predicated off still occupies the pipe for its 16 cycles, so the two kinds of step are two straight-line
// code paths selected by a warp-uniform branch.
template <int WA, int X0, int XN, bool XS>
__device__ __forceinline__ void b_step(double (&acc)[4][3][2], double (&ex)[2][2], double (&fa)[WA], double (&fb)[3], double fx,
                                       int adelta, const double *&a1, const double *&b1, int &s1, bool last, bool more_stages,
                                       const double *tA, const double *tB, const double *sAl, const double *sBl, int step,
                                       unsigned bar_full) {
  constexpr int BS = 2 * kDKC * 4;          // doubles between the B fragments of neighbouring point sub-tiles
  // ---- row 0
#pragma unroll
  for (int c = 0; c < 3; c++) dmma8x8x4(acc[0][c][0], acc[0][c][1], fa[0], fb[c]);
  if (XS && X0 == 0) dmma8x8x4(ex[0][0], ex[0][1], fa[0], fx);
  if (last) {
    // the first row of DMMAs is in the pipe: make sure the next stage has landed before reloading from it
    if (more_stages) {
      s1 = (step + 1) % kDStages;
      AIMS_HS(AIMS_TIMED(0, mbar_wait(bar_full + 8 * s1, (unsigned)((step + 1) / kDStages) & 1u)))
      a1 = sAl + (size_t)s1 * kDStage; b1 = sBl + (size_t)s1 * kDStage;
    } else {
      a1 = tA; b1 = tB;                      // nothing follows: harmless reload of this stage's first step
    }
  }
  fa[0] = a1[0];
  if (WA == 1) {
#pragma unroll
    for (int c = 0; c < 3; c++) fb[c] = b1[c * BS];
  }
  // ---- rows 1 .. WA-1
#pragma unroll
  for (int a = 1; a < WA; a++) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
      dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
      if (a == WA - 1) fb[c] = b1[c * BS];
    }
    if (XS && a >= X0 && a < X0 + XN) dmma8x8x4(ex[a - X0][0], ex[a - X0][1], fa[a], fx);
    fa[a] = a1[a * 32 + ((a & 1) ? adelta : 0)];
  }
}

template <int WA, int X0, int XN>
__device__ __forceinline__ void b_mma_kloop_t(double (&acc)[4][3][2], double (&ex)[2][2], const double *sAl, int adelta,
                                              const double *sBl, const double *sXl, int tx, int tm, int nkc, int nnz8, int &step, unsigned bar_full,
                                              unsigned bar_empty, int lane) {
  constexpr int BS = 2 * kDKC * 4;
  int s = step % kDStages;
  AIMS_HS(AIMS_TIMED(0, mbar_wait(bar_full + 8 * s, (unsigned)(step / kDStages) & 1u)))
  const double *tA = sAl + (size_t)s * kDStage, *tB = sBl + (size_t)s * kDStage;
  double fa[WA], fb[3], fx = 0.0;
#pragma unroll
  for (int a = 0; a < WA; a++) fa[a] = tA[a * 32 + ((a & 1) ? adelta : 0)];
#pragma unroll
  for (int c = 0; c < 3; c++) fb[c] = tB[c * BS];
  if (XN > 0) fx = sXl[(size_t)s * kDStage + tx * 16];
#pragma unroll 1
  for (int kc = 0; kc < nkc; kc++) {
    const int nk4 = min(kDKC, nnz8 - kc * kDKC) >> 2;
    const bool more_stages = kc + 1 < nkc;
#pragma unroll 1
    for (int t = 0; t < nk4; t++) {
      const bool last = t + 1 == nk4;
      const double *a1 = tA + (t + 1) * tm * 4, *b1 = tB + (t + 1) * 16;
      int s1 = s;
      if (XN > 0 && t == tx) b_step<WA, X0, XN, true>(acc, ex, fa, fb, fx, adelta, a1, b1, s1, last, more_stages, tA, tB, sAl, sBl, step, bar_full);
      else b_step<WA, X0, XN, false>(acc, ex, fa, fb, fx, adelta, a1, b1, s1, last, more_stages, tA, tB, sAl, sBl, step, bar_full);
      if (last) {
        if (XN > 0) fx = sXl[(size_t)s1 * kDStage + tx * 16];     // the next stage's extra B fragment (its step tx)
        tA = a1; tB = b1;
      }
    }
    // every fragment of stage s is in registers (the reloads above already read the next stage): release it
    __syncwarp();
    AIMS_HS(if (lane == 0) mbar_arrive(bar_empty + 8 * s);)
    step++;
    s = step % kDStages;
  }
}

__device__ __forceinline__ void b_mma_kloop(int wa, int x0, int xn, double (&acc)[4][3][2], double (&ex)[2][2], const double *sAl,
                                            int adelta, const double *sBl, const double *sXl, int tx, int tm, int nkc, int nnz8, int &step,
                                            unsigned bar_full, unsigned bar_empty, int lane) {
#define AIMS_B_CASE(WA, X0, XN)                                                                                   \
  case WA * 16 + X0 * 4 + XN:                                                                                      \
    b_mma_kloop_t<WA, X0, XN>(acc, ex, sAl, adelta, sBl, sXl, tx, tm, nkc, nnz8, step, bar_full, bar_empty, lane);        \
    break;
  switch (wa * 16 + (xn ? x0 : 0) * 4 + xn) {
    AIMS_B_CASE(4, 0, 0) AIMS_B_CASE(4, 0, 2) AIMS_B_CASE(4, 2, 2)
    AIMS_B_CASE(3, 0, 0) AIMS_B_CASE(3, 0, 2) AIMS_B_CASE(3, 2, 1)
    AIMS_B_CASE(2, 0, 0) AIMS_B_CASE(2, 0, 2)
    AIMS_B_CASE(1, 0, 0) AIMS_B_CASE(1, 0, 1)
    default: d_idle_kloop(nkc, step, bar_full, bar_empty, lane); break;
  }
#undef AIMS_B_CASE
}

// rows of M-tile mt when nsub sub-tiles of 8 rows are cut into n_mt M-tiles of <= 8 sub-tiles (heights differ by at most one)
__host__ __device__ inline int b_mt_start(int mt, int nsub, int n_mt) { return (int)((unsigned)(mt * nsub) / (unsigned)n_mt); }

template <bool GRAD>
__global__ void __launch_bounds__(kBThreads, 1) k_density_b(DevSys S, BatchLists L, DArgs A, int max_act) {
  const DItem it = A.items[A.order ? A.order[blockIdx.x] : blockIdx.x];
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double *sA = reinterpret_cast<double *>(smem_raw);                     // stage s: [k4][tm][4] at sA + s * kDStage
  double *sPart = sA + (size_t)kDStages * kDStage;                       // [ib][q][192]: the 4 x 3 blocks
  double *sPartX = sPart + kBSlots * 4 * 8 * kBMinSub;                   // [slot (ib, h, qx)][q][8]: the 25th point sub-tile
  unsigned long long *s_bar = reinterpret_cast<unsigned long long *>(sPartX + kBXSlots * 4 * 8);
  int *sInfo = reinterpret_cast<int *>(s_bar + 2 * kDStages);           // 16-byte aligned; [pad8(max nnz)]
  int *sLd = sInfo + pad8(A.max_nnz_pad);
  long long *sPtab = reinterpret_cast<long long *>(sLd + kMaxActive);

  const int b = it.b;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nnz = L.nnz[b], nact = L.n_act[b];
  const int nnz8 = pad8(nnz), nsub = nnz8 >> 3;
  const long long pbase = S.batch_ptr[b];
  const int np = (int)(S.batch_ptr[b + 1] - pbase), np8 = pad8(np);
  const long long boff = A.pad_off[b] - A.pad_base;
  const int p0 = it.p0, npt = it.npt;                    // this CTA's points [p0, p0+npt) of the batch (multiples of 8)
  const bool has_x = (npt >> 3) > kBMinSub;              // the CTA has a 25th point sub-tile
  const int n_mt = (nsub + 7) >> 3;                      // M-tiles of <= 8 row sub-tiles
  const double *sB = sA + 64 * kDKC;                     // stage s: [point group][16][4] at sB + s * kDStage
  const int nkc = (nnz8 + kDKC - 1) / kDKC;              // K stages per M-tile
  const long long fo = L.fn_off[b], ao = L.act_off[b];
  const long long *gptab = L.ptab + L.ptab_off[b];

  for (int i = tid; i < nnz8; i += kBThreads) sInfo[i] = i < nnz ? L.fn_info[fo + i] : -1;
  for (int i = tid; i < nact; i += kBThreads) sLd[i] = L.act_ld[ao + i];
  if (A.ptab_in_smem)
    for (int i = tid; i < nact * nact; i += kBThreads) sPtab[i] = gptab[i];
  for (int i = tid; i < kBSlots * 4 * 8 * kBMinSub + kBXSlots * 4 * 8; i += kBThreads) sPart[i] = 0.0;
  const unsigned bar_full = smem_u32(s_bar), bar_empty = bar_full + 8 * kDStages;
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kDStages; s++) {
      mbar_init(bar_full + 8 * s, (unsigned)kBProd + 1u);   // the producers' cp.async completions + the expect_tx arrival
      mbar_init(bar_empty + 8 * s, (unsigned)kBMma);
    }
    mbar_fence_init();
  }
  __syncthreads();
#ifdef AIMS_PROBE_WARP_CYCLES
  if (lane == 0) { long long *w = probe_wc(); w[0] = 0; w[1] = 0; w[2] = clock64(); }
  __syncwarp();
#endif
  const long long *ptab = A.ptab_in_smem ? sPtab : gptab;
  const double *gP = A.P + boff;

  if (warp >= kBMma) {
    // =========================================================================== producers (as in density.cuh)
#ifdef AIMS_PROBE_D_NO_HANDSHAKE
    if (warp >= kBMma) return;
#endif
    const int pl = tid - kBMma * 32;               // 0..63
    int step = 0;
#pragma unroll 1
    for (int mt = 0; mt < n_mt; mt++) {
      const int i0 = b_mt_start(mt, nsub, n_mt) * 8, tm = b_mt_start(mt + 1, nsub, n_mt) * 8 - i0;
#pragma unroll 1
      for (int kc = 0; kc < nkc; kc++, step++) {
        const int s = step % kDStages;
        if (step >= kDStages) AIMS_TIMED(0, mbar_wait(bar_empty + 8 * s, (unsigned)(step / kDStages - 1) & 1u))
        const int k0 = kc * kDKC;
#ifdef AIMS_PROBE_WARP_CYCLES
        const long long tg0 = clock64();
#endif
        if (kc == max(nkc - kDPrefetchLead, 0)) {
          // operands of this M-tile's epilogue: whole 16-row chunks are contiguous in the density layout
          const int c0 = i0 >> 4, nch = ((i0 + tm - 1) >> 4) - c0 + 1;
          for (int idx = pl; idx < nch * (GRAD ? 4 : 1); idx += kBProd) {
            const int c = c0 + (GRAD ? (idx >> 2) : idx), q = GRAD ? (idx & 3) : 0;
            const double *base = (q == 0) ? gP : A.G[q - 1] + boff;
            bulk_prefetch_l2(base + ((long long)c * (np8 >> 2) + (p0 >> 2)) * 64, (unsigned)npt * 128u);
          }
        }
        if (pl == kBProd - 1) {
          // Phi rows [k0, k0+16) of every point of the CTA: ONE contiguous segment in the density layout
          mbar_expect_tx(bar_full + 8 * s, (unsigned)npt * 128u);
          bulk_g2s(smem_u32(sB + (size_t)s * kDStage), gP + ((long long)kc * (np8 >> 2) + (p0 >> 2)) * 64, (unsigned)npt * 128u,
                   bar_full + 8 * s);
        }
        d_gather_tile(sA + (size_t)s * kDStage, A.D, i0, tm, k0, nnz, nnz8, nact, sInfo, sLd, ptab, pl, kBProd);
        cp_async_mbar_arrive_noinc(bar_full + 8 * s);
#ifdef AIMS_PROBE_WARP_CYCLES
        if (lane == 0) probe_wc()[1] += clock64() - tg0;
#endif
      }
    }
  } else {
    // =========================================================================== MMA warps
    // sub-partition = warp & 3: each hosts two warps of either row block
    const int ib = (warp >> 2) & 1, pb = (warp & 3) + 4 * (warp >> 3);
    const int xh = pb & 1, qx = pb >> 1;                   // my piece of the 25th sub-tile: row half xh, in K step tx of a stage
    const int tx = (4 - qx) & 3;
    const int ps0 = 24 * pb, px0 = 8 * kBMinSub;           // first point (within the CTA) of my block / of the 25th sub-tile
    const int fr = lane >> 2, fk = lane & 3;
    const int boffl = ((ps0 >> 2) + (fr >> 2)) * (kDKC * 4) + fk * 4 + (fr & 3);
    const int xoffl = ((px0 >> 2) + (fr >> 2)) * (kDKC * 4) + fk * 4 + (fr & 3);
    double acc[4][3][2], ex[2][2];
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
      for (int c = 0; c < 3; c++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }
    ex[0][0] = ex[0][1] = ex[1][0] = ex[1][1] = 0.0;

    int step = 0;
#pragma unroll 1
    for (int mt = 0; mt < n_mt; mt++) {
      const int m0 = b_mt_start(mt, nsub, n_mt), hm = b_mt_start(mt + 1, nsub, n_mt) - m0;   // sub-tiles
      const int i0 = m0 * 8, tm = hm * 8;
      const int wa0 = (hm + 1) >> 1;
      const int wa = ib == 0 ? wa0 : hm - wa0;             // my row block: <= 4 sub-tiles
      const int ri0 = i0 + (ib == 0 ? 0 : wa0 * 8);
      const int x0 = 2 * xh, xn = has_x ? max(0, min(2, wa - x0)) : 0;
      const int aoffl = (ri0 - i0) * 4 + lane, adelta = 0;
      b_mma_kloop(wa, x0, xn, acc, ex, sA + aoffl, adelta, sB + boffl, sB + xoffl, tx, tm, nkc, nnz8, step, bar_full, bar_empty, lane);

#ifdef AIMS_PROBE_WARP_CYCLES
      const long long te0 = clock64();
#endif
      // ---- M-tile epilogue: n_p += sum_i Phi_ip temp_ip (and gradient), rows reduced by shuffles
      constexpr int NQ = GRAD ? 4 : 1;
      // one 8-point column of accumulators av[a][0..1], a < na, rows rbase + 8 a + fr: multiply, reduce over rows, add to slot
      auto column = [&](const double (*av)[2], int na, int rbase, int col, double *part, int pstride) {
        const int p = p0 + col;                              // within the batch (even)
        double sn[2] = {0.0, 0.0}, sg[3][2] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
        for (int a0 = 0; a0 < 4; a0 += 2) {
          if (a0 < na) {
            double2 ev[2][NQ];
#pragma unroll
            for (int da = 0; da < 2; da++) {
              const int i = rbase + min(a0 + da, na - 1) * 8 + fr;   // < nnz8: padding rows are zero in the planes
              const long long o = (((long long)(i >> 4) * (np8 >> 2) + (p >> 2)) * 16 + (i & 15)) * 4 + (p & 3);
              ev[da][0] = __ldg(reinterpret_cast<const double2 *>(gP + o));
              if (GRAD)
#pragma unroll
                for (int q = 0; q < 3; q++) ev[da][q + 1] = __ldg(reinterpret_cast<const double2 *>(A.G[q] + boff + o));
            }
#pragma unroll
            for (int da = 0; da < 2; da++) {
              if (a0 + da < na) {
                sn[0] += ev[da][0].x * av[a0 + da][0];
                sn[1] += ev[da][0].y * av[a0 + da][1];
                if (GRAD)
#pragma unroll
                  for (int q = 0; q < 3; q++) {
                    sg[q][0] += ev[da][q + 1].x * av[a0 + da][0];
                    sg[q][1] += ev[da][q + 1].y * av[a0 + da][1];
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
        if (fr == 0) {   // lanes 0..3 own columns 2*fk, 2*fk+1; (slot, column) has exactly one owner warp -> no race
          double *pp = part;
          pp[0] += sn[0]; pp[1] += sn[1];
          if (GRAD)
#pragma unroll
            for (int q = 0; q < 3; q++) { pp[(q + 1) * pstride] += sg[q][0]; pp[(q + 1) * pstride + 1] += sg[q][1]; }
        }
      };
#ifdef AIMS_PROBE_NO_D_EPILOGUE
      if (wa > 0) {   // keep the accumulators live through a store that never happens
        double sum = ex[0][0] + ex[0][1] + ex[1][0] + ex[1][1];
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
          for (int c = 0; c < 3; c++) sum += acc[a][c][0] + acc[a][c][1];
        if (sum == 12345.678) sPart[lane] = sum;
      }
      if (false) {
#else
      if (wa > 0) {
#endif
#pragma unroll
        for (int c = 0; c < 3; c++) {
          double av[4][2];
#pragma unroll
          for (int a = 0; a < 4; a++) { av[a][0] = acc[a][c][0]; av[a][1] = acc[a][c][1]; }
          const int col = ps0 + c * 8 + 2 * fk;
          column(av, wa, ri0, col, sPart + (ib * 4) * (8 * kBMinSub) + col, 8 * kBMinSub);
        }
        if (xn > 0) {
          double av[4][2] = {{ex[0][0], ex[0][1]}, {ex[1][0], ex[1][1]}, {0.0, 0.0}, {0.0, 0.0}};
          column(av, xn, ri0 + x0 * 8, px0 + 2 * fk, sPartX + (((ib * 2 + xh) * 4 + qx) * 4) * 8 + 2 * fk, 8);
        }
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
          for (int c = 0; c < 3; c++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }
        ex[0][0] = ex[0][1] = ex[1][0] = ex[1][1] = 0.0;
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
           warp >= kBMma ? "prod" : "mma ", warp, clock64() - w[2], w[0], warp >= kBMma ? "gather" : "epilogue", w[1]);
  }
#endif

  // ---- S3d: store (mapping to the global point array is the identity on the batch's contiguous range)
  for (int col = tid; col < npt; col += kBThreads) {
    const int p = p0 + col;
    if (p >= np) continue;
    // sum of the partial-sum slots of plane q at this column, in a fixed order (deterministic)
    auto total = [&](int q) {
      double v = 0.0;
      if (col < 8 * kBMinSub) {
#pragma unroll
        for (int m = 0; m < kBSlots; m++) v += sPart[(m * 4 + q) * (8 * kBMinSub) + col];
      } else {
#pragma unroll
        for (int m = 0; m < kBXSlots; m++) v += sPartX[(m * 4 + q) * 8 + col - 8 * kBMinSub];
      }
      return v;
    };
    A.n[pbase + p] = total(0);
    if (GRAD)
#pragma unroll
      for (int q = 0; q < 3; q++) A.gn[(long long)q * A.n_points + pbase + p] = 2.0 * total(q + 1);
  }
}

}  // namespace aims
