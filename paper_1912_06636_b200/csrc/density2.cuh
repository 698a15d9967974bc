// density2.cuh -- S3a-S3d again (see density.cuh for the operation and its citations), in the decomposition that feeds the
// FP64 tensor pipe WITHOUT producer warps:  temp = D_b . Phi on DMMA.8x8x4, n_p = sum_i Phi_ip temp_ip, grad n likewise.
//
// What changed against density.cuh, and why (round-1 counters: 14 of 16 warps on the pipe, two producer warps gathering D_b
// with 8-byte cp.async -- 224 rows per stage for batches of <= 100 points --, all warps in their M-tile epilogue at once):
//   * "calculate_density_mat" (PAPER.md L314 / L357) is split in two.  Once per call, k_expand_matrix writes the symmetric
//     block-sparse matrix out as FULL storage (both triangles), every atom-pair block (A, B) as [pair of columns][row][2]
//     with the columns of B padded to an even count.  In that form the piece "rows r0..r1 of atom A x one column pair of
//     atom B" is a contiguous, 16-byte aligned run, whichever triangle it came from.
//   * The K order of a batch ("K''") starts every active atom at an even index (k_eval<., kLayD2> inserts a zero row after
//     an atom with an odd number of rows), so a column pair never straddles two atoms and the D_b tile of a K stage is a
//     set of 16-byte pieces with ONE table look-up each: every MMA warp copies its share of the next tile (two to four
//     cp.async of 16 bytes per lane and stage) -- no 8-byte gathers, no transposed reads, no branches, no producer warps.
//     (Issuing the runs as bulk copies, UBLKCP, from the lanes of one warp was measured first: per-lane operands of a
//     uniform-datapath instruction are serialised, ~1,500 cycles per stage: profiles/r02_kernel_experiments.md.)
//   * A CTA is 8 MMA warps on a (batch, <= 128 points) item and two CTAs share an SM: one CTA's M-tile epilogue and set-up
//     overlap the other's DMMAs, and the ragged sub-partition loads of the two CTAs (rotated by the CTA index) average out.
// Only for batches whose active atoms keep ALL their shells (true whenever the shells of a species share one cutoff, as in
// every configuration of BASELINE.json); contexts with partially culled atoms use density.cuh.
#pragma once
#include "common.cuh"
#include "density.cuh"   // DItem, blk_start / blk_count

namespace aims {

constexpr int kD2KC = 16;                 // K'' values per stage (8 pairs)
constexpr int kD2MaxStages = 4;
constexpr int kD2Threads = 288;           // 8 MMA warps + 1 producer warp; two CTAs per SM -> <= 112 registers per thread
constexpr int kD2Warps = 8;
constexpr int kD2MaxPts = 104;            // points per CTA (4 blocks of <= 32; a 200-point batch is two items of 104 + 96)
// A stage holds the D_b tile, 8 pairs x (2 tm + 8) doubles, then the Phi tile, npt x 16:
//   4 point blocks (65..104 points): tm =  64 -> 1088 + 1664 = 2752 doubles, FOUR stages;
//   1-2 point blocks (<= 64 points): tm = 128 -> 2112 + 1024 = 3136 doubles, THREE stages in the same 88 KB.
// The refill of a stage is issued one stage after its release (so that the issuing warp never waits for the slowest
// one), which leaves N - 2 stages of flight time for the copies: with three stages of 16 functions the 100-point items of
// the first version waited on the "full" barriers for 19 % of their time (ncu, profiles/r02_kernel_experiments.md).
constexpr int kD2StageDoubles4 = 2752, kD2StageDoubles3 = 3136;
constexpr int kD2SmemStageDoubles = 4 * kD2StageDoubles4;      // 11008 >= 3 * 3136
constexpr int kD2PrefetchLead = 6;

struct D2Ring {            // stage ring of a CTA: N buffers of `stride` doubles
  int n, stride;
  __device__ __forceinline__ int slot(int q) const { return n == 4 ? (q & 3) : (q % 3); }
  __device__ __forceinline__ unsigned phase(int q) const { return (unsigned)(n == 4 ? (q >> 2) : (q / 3)) & 1u; }
};

// ---- full-storage expansion of a block-sparse symmetric matrix ------------------------------------------------------
// For the upper block q = (A, B), A <= B, of the pattern:  U part = block (A, B), L part (A < B) = block (B, A) = its transpose.
// Block (X, Y) is stored as [c >> 1][row r < n_fn(X)][c & 1], c < pad2(n_fn(Y)), zero for c >= n_fn(Y).
struct ExpandArgs {
  const double *M;               // block-sparse values (upper blocks, row-major [n_fn(A)][ld])
  double *F;                     // full storage
  const long long *offU, *offL;  // [n_blocks] offsets into F (offL unused for diagonal blocks)
  const int *blk_row;            // [n_blocks] row atom of every block
  long long zero_doubles;        // F[0 .. zero_doubles) is kept zero (source of the pieces of absent blocks)
};

__global__ void __launch_bounds__(256) k_expand_matrix(DevSys S, ExpandArgs X, long long n_blocks) {
  const long long q = blockIdx.x;
  if (q >= n_blocks) return;
  const int A = X.blk_row[q], B = S.col_atom[q];
  const int nA = S.atom_fn_ptr[A + 1] - S.atom_fn_ptr[A], nB = S.atom_fn_ptr[B + 1] - S.atom_fn_ptr[B];
  const int ld = S.blk_ld[q];
  const double *src = X.M + S.blk_off[q];
  double *U = X.F + X.offU[q];
  const int nB2 = (nB + 1) & ~1, nA2 = (nA + 1) & ~1;
  for (int e = threadIdx.x; e < nA * nB2; e += 256) {              // e = r * nB2 + c: coalesced reads along c
    const int r = e / nB2, c = e - r * nB2;
    U[((c >> 1) * nA + r) * 2 + (c & 1)] = c < nB ? src[(long long)r * ld + c] : 0.0;
  }
  if (A != B) {
    double *Lp = X.F + X.offL[q];
    for (int e = threadIdx.x; e < nB * nA2; e += 256) {            // block (B, A): rows r of B, columns c of A
      const int c = e / nB, r = e - c * nB;                        // r fastest: coalesced writes along r (pairs interleaved)
      Lp[((c >> 1) * nB + r) * 2 + (c & 1)] = c < nA ? src[(long long)c * ld + r] : 0.0;
    }
  }
}

struct D2Args {
  const DItem *items;
  const int *order;
  const double *P;                  // Phi plane (kLayD2)
  const double *G[3];               // gradient planes (GRAD only)
  const long long *pad_off;         // [n_batches+1] prefix of round_up(kq,16)*pad8(np)
  long long pad_base;
  const double *F;                  // full-storage density matrix (k_expand_matrix)
  const long long *offU, *offL;
  double *n, *gn;
  long long n_points;
  int max_nnz_pad;                  // capacity of the per-row table
  int max_kq_pad;                   // capacity of the per-pair table (pairs)
  int pblk_in_smem;
};

inline size_t d2_smem_bytes(int max_nnz, int max_kq, int max_act, bool pblk_in_smem) {
  size_t s = (size_t)kD2SmemStageDoubles * sizeof(double);
  s += (size_t)4 * 256 * sizeof(double);                         // part[ib][q][col]: IB * npt <= 256
  s += 2 * kD2MaxStages * sizeof(unsigned long long);
  s += (size_t)round_up(max_nnz + 8, 16) * sizeof(unsigned short);   // sInfo
  s += (size_t)(round_up(max_kq, 16) / 2) * sizeof(unsigned char) + 16;   // slot of every K'' pair
  s += (size_t)3 * (kMaxActive + 4) * sizeof(int);               // row0, kq0, n_fn per slot
  (void)pblk_in_smem;
  s += (size_t)max_act * max_act * sizeof(unsigned);             // block offsets of every slot pair
  return s;
}

// K loop of one warp block of (8 WA rows) x (8 WB points) over nkc stages: d_mma_kloop_t of density.cuh with the A tile in the
// [pair][row][2] layout (pair stride PS = 2 tm + 8 doubles: the two halves of a fragment fall into disjoint banks).
//   A fragment a of k4-step t:  tA[(2 t) PS + a 16]   with the lane offset  (row in tile) 2 + (k & 1) + (k >> 1) PS  folded into tA.
// refill(q): called by the whole warp after it has released stage q -- the kernel's rotating refill duty.
template <int WA, int WB, class Refill>
__device__ __forceinline__ void d2_mma_kloop_t(double (&acc)[4][4][2], const double *sAl, const double *sBl, int PS, int nkc,
                                               int kq4, int &step, unsigned bar_full, unsigned bar_empty, int lane,
                                               const D2Ring R, Refill &&refill) {
  int s = R.slot(step);
  mbar_wait(bar_full + 8 * s, R.phase(step));
  const double *tA = sAl + s * R.stride, *tB = sBl + s * R.stride;
  double fa[WA], fb[WB];
#pragma unroll
  for (int a = 0; a < WA; a++) fa[a] = tA[a * 16];
#pragma unroll
  for (int c = 0; c < WB; c++) fb[c] = tB[c * (2 * kD2KC * 4)];
#pragma unroll 1
  for (int kc = 0; kc < nkc; kc++) {
    const int nk4 = min(kD2KC, kq4 - kc * kD2KC) >> 2;        // k4-steps of this stage (kq4 = K'' rows rounded up to 4)
    const bool more_stages = kc + 1 < nkc;
#pragma unroll 1
    for (int t = 0; t < nk4; t++) {
      const bool last = t + 1 == nk4;
      const double *a1 = tA + (t + 1) * 2 * PS, *b1 = tB + (t + 1) * 16;
#pragma unroll
      for (int c = 0; c < WB; c++) dmma8x8x4(acc[0][c][0], acc[0][c][1], fa[0], fb[c]);
      if (last) {
        if (more_stages) {
          const int s1 = R.slot(step + 1);
          mbar_wait(bar_full + 8 * s1, R.phase(step + 1));
          a1 = sAl + s1 * R.stride; b1 = sBl + s1 * R.stride;
        } else {
          a1 = tA; b1 = tB;
        }
      }
      if (WA > 1) {
        fa[0] = a1[0];
#pragma unroll
        for (int a = 1; a < WA - 1; a++) {
#pragma unroll
          for (int c = 0; c < WB; c++) dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
          fa[a] = a1[a * 16];
        }
#pragma unroll
        for (int c = 0; c < WB; c++) {
          dmma8x8x4(acc[WA - 1][c][0], acc[WA - 1][c][1], fa[WA - 1], fb[c]);
          fb[c] = b1[c * (2 * kD2KC * 4)];
        }
        fa[WA - 1] = a1[(WA - 1) * 16];
      } else {
        fa[0] = a1[0];
#pragma unroll
        for (int c = 0; c < WB; c++) fb[c] = b1[c * (2 * kD2KC * 4)];
      }
      if (last) { tA = a1; tB = b1; }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_empty + 8 * s);
    refill(step);
    step++;
    s = R.slot(step);
  }
}

template <class Refill>
__device__ __forceinline__ void d2_idle_kloop(int nkc, int &step, unsigned bar_full, unsigned bar_empty, int lane, const D2Ring R,
                                              Refill &&refill) {
#pragma unroll 1
  for (int kc = 0; kc < nkc; kc++, step++) {
    const int s = R.slot(step);
    mbar_wait(bar_full + 8 * s, R.phase(step));
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_empty + 8 * s);
    refill(step);
  }
}

template <class Refill>
__device__ __forceinline__ void d2_mma_kloop(int variant, double (&acc)[4][4][2], const double *sAl, const double *sBl, int PS,
                                             int nkc, int kq4, int &step, unsigned bar_full, unsigned bar_empty, int lane,
                                             const D2Ring R, Refill &&refill) {
#define AIMS_D2_CASE(WA, WB)                                                                         \
  case WA * 4 + WB:                                                                                  \
    d2_mma_kloop_t<WA, WB>(acc, sAl, sBl, PS, nkc, kq4, step, bar_full, bar_empty, lane, R, refill); \
    break;
  switch (variant) {
    AIMS_D2_CASE(4, 4) AIMS_D2_CASE(4, 3) AIMS_D2_CASE(3, 4) AIMS_D2_CASE(3, 3)
    AIMS_D2_CASE(4, 2) AIMS_D2_CASE(4, 1) AIMS_D2_CASE(3, 2) AIMS_D2_CASE(3, 1)
    AIMS_D2_CASE(2, 4) AIMS_D2_CASE(2, 3) AIMS_D2_CASE(2, 2) AIMS_D2_CASE(2, 1)
    AIMS_D2_CASE(1, 4) AIMS_D2_CASE(1, 3) AIMS_D2_CASE(1, 2) AIMS_D2_CASE(1, 1)
    default: d2_idle_kloop(nkc, step, bar_full, bar_empty, lane, R, refill); break;
  }
#undef AIMS_D2_CASE
}

// Tables of one batch in shared memory, shared by every kernel built on this pipeline.
struct D2Tables {
  const unsigned short *sInfo;   // [nnz8] (slot << 8) | row inside the atom's block (n_fn <= 224, <= 96 slots), 0xFFFF beyond nnz
  const unsigned char *sPairSlot;// [kq16 / 2] slot of every K'' pair (0xFF beyond kq)
  const int *sRow0, *sKq0, *sNfn;// [nact (+1)] first row, first K'' row, function count of every slot
  const unsigned *sPoff;         // [nact^2] offset (in 16-byte units) of block (si, sj) in the full storage, ~0u if absent
  int nact, nnz, kq;
};

// This thread's share of the D_b tile of one stage: rows [i0, i0 + tm) x K'' [16 kc, 16 kc + 16) as tm x 8 pieces of 16
// bytes (one row, one column pair); piece index = t + k * nthreads, pair = piece & 7, row = piece >> 3.  Rows beyond nnz,
// pairs beyond kq and atom pairs outside the pattern are zero-filled (src_bytes = 0).  The thread's copies arrive on `bar`
// when they have landed (cp.async.mbarrier.arrive.noinc).
__device__ __forceinline__ void d2_fill_tile(const D2Tables &T, const double *F, double *stage, unsigned bar, int i0, int tm, int kc,
                                             int t, int nthreads) {
  const int PS = 2 * tm + 8;
  const int u = t & 7;
  const int k2 = kc * kD2KC + 2 * u;                                // first K'' row of my column pair
  const int sj = k2 < T.kq ? T.sPairSlot[k2 >> 1] : -1;
  const int cp = sj >= 0 ? (k2 - T.sKq0[sj]) >> 1 : 0;              // column pair inside atom sj
  const unsigned dst0 = smem_u32(stage + u * PS);
#pragma unroll 2
  for (int r = t >> 3; r < tm; r += nthreads >> 3) {
    const unsigned fi = (i0 + r < T.nnz && sj >= 0) ? T.sInfo[i0 + r] : 0xFFFFu;
    const int si = fi >> 8, ri = fi & 0xFF;
    const double *src = F;
    int bytes = 0;
    if (fi != 0xFFFFu) {
      const unsigned po = T.sPoff[si * T.nact + sj];
      if (po != ~0u) { src = F + ((long long)po + (long long)cp * T.sNfn[si] + ri) * 2; bytes = 16; }
    }
    cp_async16(dst0 + (unsigned)r * 16u, src, bytes);
  }
  cp_async_mbar_arrive_noinc(bar);
}

template <bool GRAD>
__global__ void __maxnreg__(112) k_density2(DevSys S, BatchLists L, D2Args A, int max_act) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double *sStage = reinterpret_cast<double *>(smem_raw);
  double *sPart = sStage + kD2SmemStageDoubles;                          // [ib][q][col]
  unsigned long long *s_bar = reinterpret_cast<unsigned long long *>(sPart + 4 * 256);
  int *sRow0 = reinterpret_cast<int *>(s_bar + 2 * kD2MaxStages);
  int *sKq0 = sRow0 + (kMaxActive + 4);
  int *sNfn = sKq0 + (kMaxActive + 4);
  unsigned *sPoff = reinterpret_cast<unsigned *>(sNfn + (kMaxActive + 4));
  unsigned short *sInfo = reinterpret_cast<unsigned short *>(sPoff + max_act * max_act);
  unsigned char *sPairSlot = reinterpret_cast<unsigned char *>(sInfo + round_up(A.max_nnz_pad + 8, 16));

  const DItem it = A.items[A.order ? A.order[blockIdx.x] : blockIdx.x];
  const int b = it.b;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nnz = L.nnz[b], nact = L.n_act[b], kq = L.kq[b];
  const int nnz8 = pad8(nnz), nsub = nnz8 >> 3, nblk = blk_count(nsub);
  const long long pbase = S.batch_ptr[b];
  const int np = (int)(S.batch_ptr[b + 1] - pbase);
  const int np8 = pad8(np);
  const long long boff = A.pad_off[b] - A.pad_base;
  const int p0 = it.p0, npt = it.npt;
  const int psub = npt >> 3;
  const int PB = psub > 8 ? 4 : (psub > 4 ? 2 : 1);                // point blocks of 2..4 sub-tiles: PB x IB = 8 warps (4 for <= 32 points)
  const int IB = PB == 4 ? 2 : 4;                                  // row blocks per M-tile
  const D2Ring R{PB == 4 ? 4 : 3, PB == 4 ? kD2StageDoubles4 : kD2StageDoubles3};
  const int n_mt = (nblk + IB - 1) / IB;
  const int kq16 = round_up(kq, 16), nkc = kq16 / kD2KC, kq4 = round_up(kq, 4);
  const long long fo = L.fn_off[b], ao = L.act_off[b];
  const int *gpblk = L.pblk + L.ptab_off[b];

  for (int i = tid; i < nnz8; i += kD2Threads) {
    const int fi = i < nnz ? L.fn_info[fo + i] : -1;
    sInfo[i] = fi >= 0 ? (unsigned short)(((fi >> 16) << 8) | (fi & 0xFF)) : (unsigned short)0xFFFF;
  }
  for (int i = tid; i < nact; i += kD2Threads) sRow0[i] = L.act_row0[ao + i];
  for (int i = tid; i < nact * nact; i += kD2Threads) {
    const int si = i / nact, sj = i - si * nact;
    const int q = gpblk[i];
    sPoff[i] = q >= 0 ? (unsigned)((si <= sj ? A.offU[q] : A.offL[q]) >> 1) : ~0u;
  }
  for (int i = tid; i < 4 * 256; i += kD2Threads) sPart[i] = 0.0;
  // stale stage contents are multiplied with zero rows of Phi (K'' padding): they must be finite
  for (int i = tid; i < kD2SmemStageDoubles; i += kD2Threads) sStage[i] = 0.0;
  const unsigned bar_full = smem_u32(s_bar), bar_empty = bar_full + 8 * kD2MaxStages;
  __shared__ int s_map[kD2Warps + 1];
  __shared__ int s_nlive;
  __syncthreads();
  if (tid == 0) {
    int k0 = 0;
    for (int s = 0; s < nact; s++) {
      const int nf = (s + 1 < nact ? sRow0[s + 1] : nnz) - sRow0[s];
      sNfn[s] = nf; sKq0[s] = k0;
      k0 += (nf + 1) & ~1;
    }
    sKq0[nact] = k0; sRow0[nact] = nnz;
    // blocks (pb, ib) -> warps.  Sub-partition q hosts warps q and q + 4.  Neighbouring blocks of a row block go to
    // different sub-partitions, the next row block starts two further (the widest point block is pb = 0), and the whole
    // pattern is rotated by the CTA index, so that the ragged loads of the two CTAs of an SM fall on different FP64 pipes.
    const int rot = blockIdx.x & 3;
    int nl = 0;
    for (int w = 0; w < kD2Warps; w++) s_map[w] = -1;
    for (int ib2 = 0; ib2 < IB; ib2++)
      for (int pb2 = 0; pb2 < PB; pb2++) {
        const int q = ((PB == 1 ? ib2 : pb2 + 2 * ib2) + rot) & 3;
        int w = s_map[q] < 0 ? q : (s_map[q + 4] < 0 ? q + 4 : -1);
        if (w < 0)
          for (w = 0; s_map[w] >= 0; w++) {}                       // PB * IB <= 8: a free warp exists
        s_map[w] = pb2 | (ib2 << 8);
        nl++;
      }
    s_nlive = nl;
  }
  __syncthreads();
  for (int i = tid; i < kq16 / 2; i += kD2Threads) {
    // slot of K'' pair i: the last slot whose first K'' row is <= 2 i (binary search over <= 96 slots)
    int lo = 0, hi = nact - 1;
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (sKq0[mid] <= 2 * i) lo = mid; else hi = mid - 1; }
    sPairSlot[i] = (2 * i < kq) ? (unsigned char)lo : 0xFF;
  }
  const int nlive = s_nlive;
  if (tid == 0) {
#pragma unroll
    // full: every thread of the live warps (its cp.async pieces) + the expect_tx arrival of the Phi bulk copy
    for (int s = 0; s < kD2MaxStages; s++) { mbar_init(bar_full + 8 * s, 32u + 1u); mbar_init(bar_empty + 8 * s, (unsigned)nlive); }
    mbar_fence_init();
  }
  fence_proxy_async();            // the zero fill of the stages (generic proxy) is ordered before the bulk copies (async proxy)
  __syncthreads();

  const int wmap = warp < kD2Warps ? s_map[warp] : -1;
  D2Tables T{sInfo, sPairSlot, sRow0, sKq0, sNfn, sPoff, nact, nnz, kq};
  const double *gP = A.P + boff;
  const bool wlive = wmap >= 0;                 // warps without a block own no barrier arrival: they only join the final store
  const int wrank = 0;                          // (the producer warp is the only one that fills stages)
  const int total_steps = n_mt * nkc;
  const int tm = IB * 32, PS = 2 * tm + 8;      // fixed tile geometry (pair stride of the A tile)
  // stage q, this warp's share: its pieces of the D_b tile; live warp 0 also starts the Phi copy and the epilogue prefetch
  auto issue = [&](int q) {
    const int mt = q / nkc, kc = q - mt * nkc;
    const int bi0 = mt * IB, bi1 = min(bi0 + IB, nblk);
    const int i0 = blk_start(bi0, nsub, nblk);
    const int s = R.slot(q);
    double *stage = sStage + s * R.stride;
    const unsigned bar = bar_full + 8 * s;
    if (wrank == 0) {
      if (lane == 0) {
        // Phi rows [16 kc, 16 kc + 16) of the CTA's points: ONE contiguous segment of the plane
        mbar_expect_tx(bar, (unsigned)npt * 128u);
        bulk_g2s(smem_u32(stage + 8 * PS), gP + ((long long)kc * (np8 >> 2) + (p0 >> 2)) * 64, (unsigned)npt * 128u, bar);
      }
      if (kc == max(nkc - kD2PrefetchLead, 0)) {
        // operands of this M-tile's epilogue: the K'' rows of the tile's rows in every plane, whole 16-row chunks -> L2
        const int ia = i0, ib_ = min(blk_start(bi1, nsub, nblk), nnz) - 1;
        const int sa = sInfo[ia] >> 8, sb = sInfo[ib_] >> 8;
        const int ka = sKq0[sa] + (ia - sRow0[sa]), kb = sKq0[sb] + (ib_ - sRow0[sb]);
        const int c0 = ka >> 4, nch = (kb >> 4) - c0 + 1;
        for (int idx = lane; idx < nch * (GRAD ? 4 : 1); idx += 32) {
          const int c = c0 + (GRAD ? (idx >> 2) : idx), pl = GRAD ? (idx & 3) : 0;
          const double *base = (pl == 0) ? gP : A.G[pl - 1] + boff;
          bulk_prefetch_l2(base + ((long long)c * (np8 >> 2) + (p0 >> 2)) * 64, (unsigned)npt * 128u);
        }
      }
    }
    d2_fill_tile(T, A.F, stage, bar, i0, tm, kc, lane, 32);
  };
  auto refill = [](int) {};                     // the MMA warps never touch the copies

  if (warp == kD2Warps) {
    // =========================================================================== producer warp
#pragma unroll 1
    for (int q = 0; q < total_steps; q++) {
      if (q >= R.n) mbar_wait(bar_empty + 8 * R.slot(q), R.phase(q - R.n));
      issue(q);
    }
  } else if (wlive) {
    const int pb = wmap & 0xFF, ib = wmap >> 8;
    const int ps0 = blk_start(pb, psub, PB);
    const int wb = (blk_start(pb + 1, psub, PB) - ps0) >> 3;
    const int fr = lane >> 2, fk = lane & 3;
    const double *sB = sStage + 8 * PS;
    const int boffl = (ps0 >> 2) * (kD2KC * 4) + (fr >> 2) * (kD2KC * 4) + fk * 4 + (fr & 3);
    double acc[4][4][2];
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
      for (int c = 0; c < 4; c++) { acc[a][c][0] = 0.0; acc[a][c][1] = 0.0; }

    int step = 0;
#pragma unroll 1
    for (int mt = 0; mt < n_mt; mt++) {
      const int bi0 = mt * IB, bi1 = min(bi0 + IB, nblk);
      const int i0 = blk_start(bi0, nsub, nblk);
      const int bi = bi0 + ib;
      const bool blive = bi < bi1;
      int wa = 0, ri0 = 0;
      if (blive) { ri0 = blk_start(bi, nsub, nblk); wa = (blk_start(bi + 1, nsub, nblk) - ri0) >> 3; }
      const int variant = blive ? wa * 4 + wb : 0;
      const int aoffl = (ri0 - i0 + fr) * 2 + (fk & 1) + (fk >> 1) * PS;
      d2_mma_kloop(variant, acc, sStage + aoffl, sB + boffl, PS, nkc, kq4, step, bar_full, bar_empty, lane, R, refill);

      if (blive) {
        // ---- M-tile epilogue: n_p += sum_i Phi_ip temp_ip (and gradient), rows reduced by shuffles
#pragma unroll
        for (int c = 0; c < 4; c++) {
          if (c < wb) {
            const int col = ps0 + c * 8 + 2 * fk;
            const int p = p0 + col;
            double sn[2] = {0.0, 0.0}, sg[3][2] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
            constexpr int NQ = GRAD ? 4 : 1;
#pragma unroll
            for (int a0 = 0; a0 < 4; a0 += 2) {
              if (a0 < wa) {
                double2 ev[2][NQ];
                bool ok[2];
#pragma unroll
                for (int da = 0; da < 2; da++) {
                  const int i = ri0 + min(a0 + da, wa - 1) * 8 + fr;
                  ok[da] = i < nnz && a0 + da < wa;
                  const int ic = min(i, nnz - 1);
                  const int sl = sInfo[ic] >> 8;
                  const int k2 = sKq0[sl] + (ic - sRow0[sl]);      // K'' row of function i
                  const long long o = (((long long)(k2 >> 4) * (np8 >> 2) + (p >> 2)) * 16 + (k2 & 15)) * 4 + (p & 3);
                  ev[da][0] = __ldg(reinterpret_cast<const double2 *>(gP + o));
                  if (GRAD)
#pragma unroll
                    for (int q = 0; q < 3; q++) ev[da][q + 1] = __ldg(reinterpret_cast<const double2 *>(A.G[q] + boff + o));
                }
#pragma unroll
                for (int da = 0; da < 2; da++) {
                  if (ok[da]) {
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
            if (fr == 0) {   // (ib, column) has exactly one owner warp -> no race, fixed order -> bitwise reproducible
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
    }
  }
  __syncthreads();

  // ---- S3d: store
  for (int col = tid; col < npt; col += kD2Threads) {
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

}  // namespace aims
