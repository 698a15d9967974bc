// basis.cuh -- S1a (active-function culling, nnz(B): PAPER.md L235) and S1b (basis evaluation, "calculate_phi":
// PAPER.md L314/L322/L356) on the GPU.  The paper keeps this stage on the CPU (L381); here it is two kernels.
#pragma once
#include <algorithm>

#include "common.cuh"

namespace aims {

// ---------------------------------------------------------------------------------------------------------------
// k_cull: one CTA per batch.
//   1. bounding box of the batch's points
//   2. atoms whose largest cutoff sphere may reach the box (conservative)            -> candidate list (smem)
//   3. exact test per candidate: min_p d2(p, atom) in separately rounded IEEE ops (reading P6), one warp per atom;
//      shell s touches the batch iff min d2 < rcut_s^2 (strict)                       -> shell bit mask
//   4. active atoms in ascending order (rank sort), rows per slot, nnz(B)
//   5. (not in the dry run) function lists, slot tables and the atom-pair offset table of the batch
// dry != 0: only nnz[b], n_act[b] are written (used once at context creation to size every list).
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_cull(DevSys S, BatchLists L, int b_first, int dry) {
  const int b = b_first + blockIdx.x;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long p0 = S.batch_ptr[b];
  const int np = (int)(S.batch_ptr[b + 1] - p0);

  __shared__ double s_red[8][6];
  __shared__ double s_box[6];
  __shared__ int s_ncand, s_nact, s_nnz;
  __shared__ int s_cand[kMaxCand];
  __shared__ unsigned s_cmask[kMaxCand];
  __shared__ int s_act_atom[kMaxActive];
  __shared__ unsigned s_act_mask[kMaxActive];
  __shared__ int s_act_row0[kMaxActive];

  if (tid == 0) { s_ncand = 0; s_nact = 0; s_nnz = 0; }

  // 1. bounding box
  double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
  for (int p = tid; p < np; p += 256) {
    double x = S.px[p0 + p], y = S.py[p0 + p], z = S.pz[p0 + p];
    lo[0] = fmin(lo[0], x); hi[0] = fmax(hi[0], x);
    lo[1] = fmin(lo[1], y); hi[1] = fmax(hi[1], y);
    lo[2] = fmin(lo[2], z); hi[2] = fmax(hi[2], z);
  }
#pragma unroll
  for (int c = 0; c < 3; c++)
    for (int o = 16; o > 0; o >>= 1) {
      lo[c] = fmin(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], o));
      hi[c] = fmax(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], o));
    }
  if (lane == 0)
    for (int c = 0; c < 3; c++) { s_red[warp][c] = lo[c]; s_red[warp][3 + c] = hi[c]; }
  __syncthreads();
  if (tid < 6) {
    double v = s_red[0][tid];
    for (int w2 = 1; w2 < 8; w2++) v = (tid < 3) ? fmin(v, s_red[w2][tid]) : fmax(v, s_red[w2][tid]);
    s_box[tid] = v;
  }
  __syncthreads();

  // 2. candidates: distance from the atom to the box, against the species' largest cutoff (with slack)
  if (np > 0)
    for (int a = tid; a < S.n_atoms; a += 256) {
      double q = 0.0;
#pragma unroll
      for (int c = 0; c < 3; c++) {
        double x = S.atom_xyz[3 * a + c];
        double e = fmax(fmax(s_box[c] - x, x - s_box[3 + c]), 0.0);
        q += e * e;
      }
      if (q <= S.sp_rcmax2[S.atom_species[a]] * (1.0 + 1e-9)) {
        int k = atomicAdd(&s_ncand, 1);
        if (k < kMaxCand) s_cand[k] = a;
      }
    }
  __syncthreads();
  int ncand = s_ncand;
  if (ncand > kMaxCand) { if (tid == 0) atomicExch(L.error_flag, 1); ncand = kMaxCand; }

  // 3. exact test, one warp per candidate
  for (int c = warp; c < ncand; c += 8) {
    const int a = s_cand[c];
    const double X = S.atom_xyz[3 * a], Y = S.atom_xyz[3 * a + 1], Z = S.atom_xyz[3 * a + 2];
    double dmin = 1e300;
    for (int p = lane; p < np; p += 32) {
      double dx = S.px[p0 + p] - X, dy = S.py[p0 + p] - Y, dz = S.pz[p0 + p] - Z;
      double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
      dmin = fmin(dmin, d2);
    }
    for (int o = 16; o > 0; o >>= 1) dmin = fmin(dmin, __shfl_xor_sync(0xffffffffu, dmin, o));
    if (lane == 0) {
      const int sp = S.atom_species[a];
      const int s0 = S.sp_shell_ptr[sp], s1 = S.sp_shell_ptr[sp + 1];
      unsigned m = 0;
      for (int s = s0; s < s1; s++)
        if (dmin < S.shell_rc2[s]) m |= 1u << (s - s0);
      s_cmask[c] = m;
      if (m) atomicAdd(&s_nact, 1);
    }
  }
  __syncthreads();
  const int nact = s_nact;
  if (nact > kMaxActive) {
    if (tid == 0) { atomicExch(L.error_flag, 2); L.nnz[b] = 0; L.n_act[b] = nact; }
    return;
  }

  // 4. ascending order of the active atoms (rank sort over the small candidate list)
  for (int c = tid; c < ncand; c += 256)
    if (s_cmask[c]) {
      const int a = s_cand[c];
      int rank = 0;
      for (int c2 = 0; c2 < ncand; c2++) rank += (s_cmask[c2] != 0 && s_cand[c2] < a);
      s_act_atom[rank] = a;
      s_act_mask[rank] = s_cmask[c];
    }
  __syncthreads();
  if (tid == 0) {
    int row = 0, kq = 0, nfull = 0;
    for (int s = 0; s < nact; s++) {
      s_act_row0[s] = row;
      const int a = s_act_atom[s];
      const int sp = S.atom_species[a];
      const int s0 = S.sp_shell_ptr[sp], s1 = S.sp_shell_ptr[sp + 1];
      for (int sh = s0; sh < s1; sh++)
        if (s_act_mask[s] >> (sh - s0) & 1u) row += 2 * S.shell_l[sh] + 1;
      kq += (row - s_act_row0[s] + 1) & ~1;
      nfull += S.atom_fn_ptr[a + 1] - S.atom_fn_ptr[a];
    }
    s_nnz = row;
    if (dry) {
      L.nnz[b] = row; L.n_act[b] = nact;
#ifdef AIMS_WITH_VARIANTS
      L.kq[b] = kq; L.nfull[b] = nfull;                 // density2.cuh only (probe builds)
#else
      (void)kq; (void)nfull;
#endif
    }
  }
  __syncthreads();
  if (dry) return;

  // 5. lists.  Offsets were fixed by the dry run; the counts must agree.
  const long long fo = L.fn_off[b], ao = L.act_off[b], po = L.ptab_off[b];
  if ((long long)s_nnz != L.fn_off[b + 1] - fo || (long long)nact != L.act_off[b + 1] - ao) {
    if (tid == 0) atomicExch(L.error_flag, 3);
    return;
  }
  if (tid == 0) { L.nnz[b] = s_nnz; L.n_act[b] = nact; }
  for (int s = tid; s < nact; s += 256) {
    const int a = s_act_atom[s];
    L.act_atom[ao + s] = a;
    L.act_mask[ao + s] = s_act_mask[s];
    L.act_row0[ao + s] = s_act_row0[s];
    L.act_ld[ao + s] = S.blk_ld[S.row_ptr[a]];   // diagonal block (a,a) is the first block of row a
    const int sp = S.atom_species[a];
    const int s0 = S.sp_shell_ptr[sp], s1 = S.sp_shell_ptr[sp + 1];
    int row = s_act_row0[s], local = 0;
    for (int sh = s0; sh < s1; sh++) {
      const int nm = 2 * S.shell_l[sh] + 1;
      if (s_act_mask[s] >> (sh - s0) & 1u)
        for (int m = 0; m < nm; m++, row++) {
          L.fn_index[fo + row] = S.atom_fn_ptr[a] + local + m;
          L.fn_info[fo + row] = (s << 16) | (local + m);
        }
      local += nm;
    }
  }
  for (int q = tid; q < nact * nact; q += 256) {
    const int sa = q / nact, sb = q - sa * nact;
    const int A = s_act_atom[min(sa, sb)], B = s_act_atom[max(sa, sb)];
    long long lo2 = S.row_ptr[A], hi2 = S.row_ptr[A + 1] - 1, found = -1, fidx = -1;
    while (lo2 <= hi2) {
      long long mid = (lo2 + hi2) >> 1;
      int cb = S.col_atom[mid];
      if (cb == B) { found = S.blk_off[mid]; fidx = mid; break; }
      if (cb < B) lo2 = mid + 1; else hi2 = mid - 1;
    }
    L.ptab[po + q] = found;
#ifdef AIMS_WITH_VARIANTS
    L.pblk[po + q] = (int)fidx;                         // density2.cuh only (probe builds)
#endif
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Real solid harmonics S_lm (orthonormal real Y_lm on the unit sphere, m = -l..l, no Condon-Shortley phase)
// and their Cartesian gradients, l <= 3, as explicit polynomials with literal constants.
// ---------------------------------------------------------------------------------------------------------------
template <bool GRAD>
__device__ __forceinline__ void solid_harmonics(int l, double x, double y, double z, double *Y, double *gx, double *gy,
                                                double *gz) {
  if (l == 0) {
    Y[0] = 0.28209479177387814;
    if (GRAD) { gx[0] = 0.0; gy[0] = 0.0; gz[0] = 0.0; }
  } else if (l == 1) {
    const double c = 0.4886025119029199;
    Y[0] = c * y; Y[1] = c * z; Y[2] = c * x;
    if (GRAD) {
      gx[0] = 0.0; gy[0] = c;   gz[0] = 0.0;
      gx[1] = 0.0; gy[1] = 0.0; gz[1] = c;
      gx[2] = c;   gy[2] = 0.0; gz[2] = 0.0;
    }
  } else if (l == 2) {
    const double a = 1.0925484305920792, bq = 0.31539156525252005, c = 0.5462742152960396;
    const double xx = x * x, yy = y * y, zz = z * z;
    Y[0] = a * (x * y);
    Y[1] = a * (y * z);
    Y[2] = bq * (2.0 * zz - xx - yy);
    Y[3] = a * (x * z);
    Y[4] = c * (xx - yy);
    if (GRAD) {
      gx[0] = a * y;          gy[0] = a * x;          gz[0] = 0.0;
      gx[1] = 0.0;            gy[1] = a * z;          gz[1] = a * y;
      gx[2] = -2.0 * bq * x;  gy[2] = -2.0 * bq * y;  gz[2] = 4.0 * bq * z;
      gx[3] = a * z;          gy[3] = 0.0;            gz[3] = a * x;
      gx[4] = 2.0 * c * x;    gy[4] = -2.0 * c * y;   gz[4] = 0.0;
    }
  } else {
    const double a = 0.5900435899266435, bq = 2.890611442640554, c = 0.4570457994644658, d = 0.3731763325901154,
                 e = 1.445305721320277;
    const double xx = x * x, yy = y * y, zz = z * z;
    const double q = 4.0 * zz - xx - yy;
    Y[0] = a * y * (3.0 * xx - yy);
    Y[1] = bq * x * y * z;
    Y[2] = c * y * q;
    Y[3] = d * z * (2.0 * zz - 3.0 * xx - 3.0 * yy);
    Y[4] = c * x * q;
    Y[5] = e * z * (xx - yy);
    Y[6] = a * x * (xx - 3.0 * yy);
    if (GRAD) {
      gx[0] = 6.0 * a * x * y;          gy[0] = 3.0 * a * (xx - yy);      gz[0] = 0.0;
      gx[1] = bq * y * z;               gy[1] = bq * x * z;               gz[1] = bq * x * y;
      gx[2] = -2.0 * c * x * y;         gy[2] = c * (q - 2.0 * yy);       gz[2] = 8.0 * c * y * z;
      gx[3] = -6.0 * d * x * z;         gy[3] = -6.0 * d * y * z;         gz[3] = 3.0 * d * (2.0 * zz - xx - yy);
      gx[4] = c * (q - 2.0 * xx);       gy[4] = -2.0 * c * x * y;         gz[4] = 8.0 * c * x * z;
      gx[5] = 2.0 * e * x * z;          gy[5] = -2.0 * e * y * z;         gz[5] = e * (xx - yy);
      gx[6] = 3.0 * a * (xx - yy);      gy[6] = -6.0 * a * x * y;         gz[6] = 0.0;
    }
  }
}

// Output modes of k_eval
enum EvalMode {
  kEvalPhi = 0,      // plane0 = Phi                                   (density, LDA; API without gradient)
  kEvalPhiGrad = 1,  // plane0 = Phi, planes 1..3 = d/dx, d/dy, d/dz   (density with grad n; API with gradient)
  kEvalHLda = 2,     // plane0 = Phi, plane1 = w v Phi                 (S2a fused: Eq. 25 "K = w phi" times v)
  kEvalHGga = 3,     // plane0 = Phi, plane1 = w (v/2 Phi + g . grad Phi)
  // Pulay forces (forces.cuh; Eq. 16, 18 L137-150): plane0 = Phi, plane1 = L = v Phi (+ g . grad Phi),
  // planes 2..4 = w d/dx_c Phi, and with the GGA term planes 5..7 = w (Hess Phi g)_c
  kEvalForceLda = 4,
  kEvalForceGga = 5,
  // full h_KS phi with the kinetic operator (Eq. 26, Fig. 6a "h_times_phi"):
  // plane0 = Phi, plane1 = w ((v Phi - 1/2 lap Phi) / 2 [+ g . grad Phi]) -- the SYR2K form P Q^T + Q P^T then gives
  // 1/2 [phi_i (h phi_j) + (h phi_i) phi_j], Fig. 6a's DSYR2K with alpha = 1/2
  kEvalHKinLda = 6,
  kEvalHKinGga = 7,
  // Hessian of the density (hessian.cuh): plane0 = Phi, planes 1..3 = d/dx_c Phi,
  // planes 4..9 = d_c d_e Phi in the order (xx, yy, zz, xy, xz, yz)
  kEvalHess = 8,
  // meta-GGA tau matrix (reading P1c): plane0 = [d_x Phi | d_y Phi | d_z Phi] stacked along the
  // points (kLayH with 3 x the padded points), plane1 = w xi / 2 times plane0; E.v carries xi
  kEvalTau = 9
};
__host__ __device__ constexpr int eval_planes(int mode) {
  return mode == kEvalPhi ? 1 : mode == kEvalPhiGrad ? 4 : mode == kEvalForceLda ? 5 : mode == kEvalForceGga ? 8 : mode == kEvalHess ? 10 : 2;
}

struct EvalArgs {
  double *plane[10];
  // kLayH, the k4 layout of common.cuh: element (row, p) of batch b at
  //   plane[q] + (pad_off[b] - pad_base) + ((p >> 2) * pad8(nnz) + row) * 4 + (p & 3); rows in [nnz, pad8(nnz)) and
  //   points in [n_p, pad8(n_p)) are written as zeros; a batch occupies pad8(nnz) * pad8(n_p) doubles per plane.
  // kLayD, chunks of 16 rows: (((row >> 4) * (np8 >> 2) + (p >> 2)) * 16 + (row & 15)) * 4 + (p & 3),
  //   rows padded with zeros to a multiple of 16; a batch occupies round_up(nnz,16) * pad8(n_p) doubles per plane
  const long long *pad_off;
  long long pad_base;
  // kLayApi: phi at plane[0] + (api_off[b]-api_base) + row*np + p,
  //          dphi component c at plane[1] + 3*(api_off[b]-api_base) + (c*nnz + row)*np + p
  const long long *api_off;
  long long api_base;
  const double *v, *g;   // [n_points], [3][n_points]
  long long n_points;
  int point_pad;         // kLayH only: zero columns up to this multiple of points (0 = 8; 16 for the LDA Hamiltonian planes)
  int kinetic;           // force modes only: L also carries -1/2 lap Phi (h_KS phi of Eq. 16 with the kinetic operator)
};

// ---------------------------------------------------------------------------------------------------------------
// (Hess S_lm) g for the solid harmonics above (second derivatives of the same polynomials), l <= 3: hx,hy,hz[m].
// Used by the Pulay-force planes (Eq. 18: the GGA term needs nabla_at grad phi).
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void solid_hessian_dot(int l, double x, double y, double z, double px, double py, double pz,
                                                  double *hx, double *hy, double *hz) {
  if (l < 2) {
#pragma unroll
    for (int m = 0; m < 3; m++) { hx[m] = 0.0; hy[m] = 0.0; hz[m] = 0.0; }
  } else if (l == 2) {
    const double a = 1.0925484305920792, bq = 0.31539156525252005, c = 0.5462742152960396;
    hx[0] = a * py;            hy[0] = a * px;            hz[0] = 0.0;
    hx[1] = 0.0;               hy[1] = a * pz;            hz[1] = a * py;
    hx[2] = -2.0 * bq * px;    hy[2] = -2.0 * bq * py;    hz[2] = 4.0 * bq * pz;
    hx[3] = a * pz;            hy[3] = 0.0;               hz[3] = a * px;
    hx[4] = 2.0 * c * px;      hy[4] = -2.0 * c * py;     hz[4] = 0.0;
  } else {
    const double a = 0.5900435899266435, bq = 2.890611442640554, c = 0.4570457994644658, d = 0.3731763325901154,
                 e = 1.445305721320277;
    const double xy = y * px + x * py, xz = z * px + x * pz, yz = z * py + y * pz;   // symmetric pair products
    const double dxy = x * px - y * py;
    hx[0] = 6.0 * a * xy;                                    hy[0] = 6.0 * a * dxy;                                   hz[0] = 0.0;
    hx[1] = bq * yz;                                         hy[1] = bq * xz;                                         hz[1] = bq * xy;
    hx[2] = -2.0 * c * xy;                                   hy[2] = c * (-2.0 * x * px - 6.0 * y * py + 8.0 * z * pz); hz[2] = 8.0 * c * yz;
    hx[3] = -6.0 * d * xz;                                   hy[3] = -6.0 * d * yz;                                   hz[3] = d * (-6.0 * x * px - 6.0 * y * py + 12.0 * z * pz);
    hx[4] = c * (-6.0 * x * px - 2.0 * y * py + 8.0 * z * pz); hy[4] = -2.0 * c * xy;                                 hz[4] = 8.0 * c * xz;
    hx[5] = 2.0 * e * xz;                                    hy[5] = -2.0 * e * yz;                                   hz[5] = 2.0 * e * dxy;
    hx[6] = 6.0 * a * dxy;                                   hy[6] = -6.0 * a * xy;                                   hz[6] = 0.0;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// k_eval: one CTA per batch, one thread per point.
//   set-up   the batch's active shells become a flat list in shared memory: (slot, l, first row, spline row, rcut^2)
//   per point walk the list: geometry and ONE log per (point, atom) when the slot changes, solid harmonics once per l,
//            one spline Horner per shell, then 2l+1 values per output plane.
// The output layout is a template parameter, so that an element address is one 32-bit multiply-add on a per-plane base
// pointer: kLayApi (aims_gpu_eval_basis: [row][point]), kLayH (k4 layout of hamiltonian.cuh), kLayD (k4 layout in chunks
// of 16 rows of density.cuh / forces.cuh).  In the k4 layouts the four threads of a 4-point group write one full 32-byte
// sector per row; in the API layout stores are coalesced along the point index.
// ---------------------------------------------------------------------------------------------------------------
// kLayD2 (density2.cuh): kLayD with the rows in "K'' order" -- every active atom's rows start at an even row, i.e. one zero
// row follows an atom with an odd number of rows -- so that a pair of consecutive rows never straddles two atoms.
enum EvalLayout { kLayApi = 0, kLayH = 1, kLayD = 2, kLayD2 = 3 };

#ifndef AIMS_EVAL_CTAS_PER_SM
#define AIMS_EVAL_CTAS_PER_SM 2
#endif
// Threads of a k_eval CTA.  Measured on config 5 (profiles/r02_kernel_experiments.md): 224 threads (7 warps cover a 200-point batch
// in one pass, 144 registers per thread at two CTAs per SM) are SLOWER than 256 (82.9 vs 63.2 ms per step) -- the kernel lives
// on warps in flight, not on registers per thread.  The spline coefficients (a gather through L1/L2 per point and shell, the
// largest stall of the round-1 kernel: long scoreboard 25 % / 46 % of the samples) are fetched one shell ahead.
#ifndef AIMS_EVAL_THREADS
#define AIMS_EVAL_THREADS 256
#endif
constexpr int kEvalThreads = AIMS_EVAL_THREADS;
// registers per thread: two CTAs of 7 warps per SM -> 65,536 / 448 = 146 (ptxas rounds a launch bound of 224 threads up to
// 256, hence __maxnreg__ instead); the force and Hessian planes need more and run one CTA per SM
__host__ __device__ constexpr int eval_max_regs(int mode) { return (mode == 4 || mode == 5 || mode == 8) ? 255 : (kEvalThreads <= 224 ? 144 : 128); }
#ifndef AIMS_EVAL_PREFETCH
#define AIMS_EVAL_PREFETCH 1
#endif
// dynamic shared memory of k_eval: one entry per active shell of the batch (<= nnz(B) of them)
inline size_t eval_smem_bytes(int max_nnz) { return (size_t)std::max(max_nnz, 1) * (sizeof(int2) + sizeof(double)); }

template <int LAYOUT>
__device__ __forceinline__ int eval_row_off(int row, int np, int np8) {
  // offset of (row, point 0-of-thread) relative to the thread's point base
  if (LAYOUT == kLayApi) return row * np;
  if (LAYOUT == kLayH) return row * 4;
  return row * 4 + (row >> 4) * (np8 * 16 - 64);
}

template <int MODE, int LAYOUT>
__global__ void __maxnreg__(eval_max_regs(MODE))
k_eval(DevSys S, BatchLists L, EvalArgs E, int b_first, int max_ent) {
  constexpr bool FORCE = (MODE == kEvalForceLda || MODE == kEvalForceGga);
  constexpr bool HESS = (MODE == kEvalForceGga);
  constexpr bool KIN = (MODE == kEvalHKinLda || MODE == kEvalHKinGga);
  constexpr bool FULLH = (MODE == kEvalHess);        // all six second derivatives of every function
  constexpr bool TAU = (MODE == kEvalTau);
  constexpr bool GRAD = (MODE == kEvalPhiGrad || MODE == kEvalHGga || MODE == kEvalHKinGga || FORCE || FULLH || TAU);
  constexpr int NPL = eval_planes(MODE);
  const int b = b_first + blockIdx.x;
  const int tid = threadIdx.x;
  const long long p0 = S.batch_ptr[b];
  const int np = (int)(S.batch_ptr[b + 1] - p0);
  const int nnz = L.nnz[b], nact = L.n_act[b];
  if (nnz == 0 || np == 0) return;
  const long long ao = L.act_off[b];

  extern __shared__ __align__(16) unsigned char eval_smem[];
  double *s_rc2 = reinterpret_cast<double *>(eval_smem);                 // [n_ent]
  int2 *s_ent = reinterpret_cast<int2 *>(s_rc2 + max_ent);                // [n_ent] x = slot | l << 8 | row << 12, y = spline row
  __shared__ double s_ax[kMaxActive], s_ay[kMaxActive], s_az[kMaxActive];
  __shared__ int s_e0[kMaxActive + 1];
  __shared__ int s_shift[LAYOUT == kLayD2 ? kMaxActive : 1];      // kLayD2: zero rows inserted before the slot
  __shared__ int s_zrow[LAYOUT == kLayD2 ? kMaxActive : 1];       // kLayD2: the inserted zero rows (K'' numbering)
  __shared__ int s_nz;
  const int nk1 = S.n_knots - 1;
  for (int s = tid; s < nact; s += kEvalThreads) {
    const int a = L.act_atom[ao + s];
    s_ax[s] = S.atom_xyz[3 * a]; s_ay[s] = S.atom_xyz[3 * a + 1]; s_az[s] = S.atom_xyz[3 * a + 2];
    s_e0[s + 1] = __popc(L.act_mask[ao + s]);
  }
  __syncthreads();
  if (tid == 0) {
    int e = 0;
    s_e0[0] = 0;
    for (int s = 0; s < nact; s++) { const int c = s_e0[s + 1]; s_e0[s] = e; e += c; }
    s_e0[nact] = e;
    if (LAYOUT == kLayD2) {
      int shift = 0, nz = 0;
      for (int s = 0; s < nact; s++) {
        const int r0 = L.act_row0[ao + s], r1 = s + 1 < nact ? L.act_row0[ao + s + 1] : nnz;
        s_shift[s] = shift;
        if ((r1 - r0) & 1) { s_zrow[nz++] = r1 + shift; shift++; }
      }
      s_nz = nz;
    }
  }
  __syncthreads();
  const int n_ent = s_e0[nact];
  if (n_ent > max_ent) { if (tid == 0) atomicExch(L.error_flag, 4); return; }
  for (int s = tid; s < nact; s += kEvalThreads) {
    const int a = L.act_atom[ao + s];
    const int sp = S.atom_species[a];
    const int s0 = S.sp_shell_ptr[sp], s1 = S.sp_shell_ptr[sp + 1];
    const unsigned mask = L.act_mask[ao + s];
    int row = L.act_row0[ao + s] + (LAYOUT == kLayD2 ? s_shift[s] : 0), e = s_e0[s];
    for (int sh = s0; sh < s1; sh++) {
      if (!(mask >> (sh - s0) & 1u)) continue;
      const int l = S.shell_l[sh];
      s_ent[e] = make_int2(s | (l << 8) | (row << 12), S.shell_spline[sh] * nk1);
      s_rc2[e] = S.shell_rc2[sh];
      row += 2 * l + 1;
      e++;
    }
  }
  __syncthreads();

  const int nnz8 = pad8(nnz), np8 = pad8(np);
  // points this CTA writes (k4 layouts: zero columns up to the padded point count)
  const int npx = LAYOUT == kLayApi ? np : (LAYOUT == kLayH && E.point_pad > 8 ? round_up(np, E.point_pad) : np8);
  const int nkq = LAYOUT == kLayD2 ? nnz + s_nz : nnz;                                       // kLayD2: rows incl. the inserted ones
  const int nrows = LAYOUT == kLayApi ? nnz : (LAYOUT == kLayD || LAYOUT == kLayD2 ? round_up(nkq, 16) : nnz8);   // rows this CTA writes
  double *o[NPL];
  if (LAYOUT == kLayApi) {
    const long long off = E.api_off[b] - E.api_base;
    o[0] = E.plane[0] + off;
    const long long cstride = (long long)nnz * np;
#pragma unroll
    for (int q = 1; q < NPL; q++) o[q] = E.plane[1] + 3 * off + (q - 1) * cstride;
  } else {
    const long long off = (E.pad_off[b] - E.pad_base) * (TAU ? 3 : 1);
#pragma unroll
    for (int q = 0; q < NPL; q++) o[q] = E.plane[q] + off;
  }
  const int cstr = TAU ? npx * nnz8 : 0;          // kEvalTau: distance between the d_x, d_y, d_z parts of a plane

  for (int p = tid; p < npx; p += kEvalThreads) {
    // the thread's point base inside the batch's plane; element (row, p) at pbase + eval_row_off(row)
    const int pbase = LAYOUT == kLayApi ? p : (LAYOUT == kLayH ? (p >> 2) * nnz8 * 4 + (p & 3) : (p >> 2) * 64 + (p & 3));   // kLayD, kLayD2
    double *op[NPL];
#pragma unroll
    for (int q = 0; q < NPL; q++) op[q] = o[q] + pbase;
#define AIMS_EZERO(idx)                                                  \
  {                                                                      \
    const int o_ = (idx);                                                \
    _Pragma("unroll") for (int q_ = 0; q_ < NPL; q_++) {                 \
      op[q_][o_] = 0.0;                                                  \
      if (TAU) { op[q_][o_ + cstr] = 0.0; op[q_][o_ + 2 * cstr] = 0.0; } \
    }                                                                    \
  }
    if (p >= np) {  // zero padding columns (k4 layouts only)
      for (int r = 0; r < nrows; r++) AIMS_EZERO(eval_row_off<LAYOUT>(r, np, np8))
      continue;
    }
    for (int r = nkq; r < nrows; r++) AIMS_EZERO(eval_row_off<LAYOUT>(r, np, np8))   // zero padding rows
    if (LAYOUT == kLayD2)
      for (int q = 0; q < s_nz; q++) AIMS_EZERO(eval_row_off<LAYOUT>(s_zrow[LAYOUT == kLayD2 ? q : 0], np, np8))
    const double x = S.px[p0 + p], y = S.py[p0 + p], z = S.pz[p0 + p];
    double wv = 0.0, wgx = 0.0, wgy = 0.0, wgz = 0.0, w = 0.0;
    if (MODE == kEvalHLda) wv = S.w[p0 + p] * E.v[p0 + p];
    if (TAU) wv = 0.5 * S.w[p0 + p] * E.v[p0 + p];             // w xi / 2
    if (MODE == kEvalHKinLda) { w = S.w[p0 + p]; wv = 0.5 * w * E.v[p0 + p]; }
    if (MODE == kEvalHGga || MODE == kEvalHKinGga) {
      w = S.w[p0 + p];
      wv = 0.5 * w * E.v[p0 + p];
      wgx = w * E.g[p0 + p]; wgy = w * E.g[E.n_points + p0 + p]; wgz = w * E.g[2 * E.n_points + p0 + p];
    }
    if (FORCE) {   // here wv = v and (wgx, wgy, wgz) = g, unweighted; the weight multiplies the epilogue planes
      w = S.w[p0 + p];
      wv = E.v[p0 + p];
      if (HESS) { wgx = E.g[p0 + p]; wgy = E.g[E.n_points + p0 + p]; wgz = E.g[2 * E.n_points + p0 + p]; }
    }
    int cur = -1, lcur = -1, k = 0;
    double2 c01 = make_double2(0.0, 0.0), c23 = make_double2(0.0, 0.0);   // spline coefficients of the current entry
    double d2 = 0.0, ux = 0.0, uy = 0.0, uz = 1.0, dd = 1.0, inv_dd = 1.0, xs = 0.0, ug = 0.0;
    double Y[7], gx[7], gy[7], gz[7];
    double hx[HESS ? 7 : 1], hy[HESS ? 7 : 1], hz[HESS ? 7 : 1];
    double s2[FULLH ? 6 : 1][FULLH ? 7 : 1];        // Hess S_lm at the unit vector: (xx, yy, zz, xy, xz, yz)
#pragma unroll 1
    for (int e = 0; e < n_ent; e++) {
      const int2 en = s_ent[e];
      const int slot = en.x & 0xFF, l = (en.x >> 8) & 3, row = en.x >> 12;
      if (slot != cur) {
        cur = slot; lcur = -1;
        const double dx = x - s_ax[slot], dy = y - s_ay[slot], dz = z - s_az[slot];
        d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
        const double d = sqrt(d2);
        ux = 0.0; uy = 0.0; uz = 1.0;
        if (d > 0.0) { const double inv = 1.0 / d; ux = dx * inv; uy = dy * inv; uz = dz * inv; }
        dd = fmax(d, S.r0);
        const double t = log(dd / S.r0) / S.log_inc;
        k = (int)floor(t);
        k = max(0, min(k, S.n_knots - 2));
        xs = t - (double)k;
        inv_dd = 1.0 / dd;
        if (HESS) ug = ux * wgx + uy * wgy + uz * wgz;
        // first shell of a new atom: its coefficients cannot be fetched earlier (k is only known now)
        const double2 *cf0 = reinterpret_cast<const double2 *>(S.spline_coef + (long long)(en.y + k) * 4);
        c01 = __ldg(cf0); c23 = __ldg(cf0 + 1);
      }
      // the next entry's coefficients, one iteration ahead (same atom -> same knot interval k); consumed at the loop's end
      double2 n01 = c01, n23 = c23;
      if (AIMS_EVAL_PREFETCH && e + 1 < n_ent) {
        const int2 en1 = s_ent[e + 1];
        if ((en1.x & 0xFF) == cur) {
          const double2 *cf1 = reinterpret_cast<const double2 *>(S.spline_coef + (long long)(en1.y + k) * 4);
          n01 = __ldg(cf1); n23 = __ldg(cf1 + 1);
        }
      }
      const int nm = 2 * l + 1;
      const int ro = eval_row_off<LAYOUT>(row, np, np8);
      // offset of row + m: rows of one shell may straddle a 16-row chunk boundary in the D layout
      const int mstep = LAYOUT == kLayApi ? np : 4;
      const int wrap = (LAYOUT == kLayD || LAYOUT == kLayD2) ? 16 - (row & 15) : 8;          // first m that lies in the next chunk
      const int jump = (LAYOUT == kLayD || LAYOUT == kLayD2) ? np8 * 16 - 64 : 0;
      if (d2 < s_rc2[e]) {
        if (l != lcur) {
          solid_harmonics<GRAD>(l, ux, uy, uz, Y, gx, gy, gz);
          if constexpr (HESS) solid_hessian_dot(l, ux, uy, uz, wgx, wgy, wgz, hx, hy, hz);
          if constexpr (FULLH) {
            // columns of Hess S_lm = (Hess S_lm) e_c for the three unit vectors e_c
            double t0[7], t1[7], t2[7];
            solid_hessian_dot(l, ux, uy, uz, 1.0, 0.0, 0.0, s2[0], t1, t2);       // xx, (yx), (zx)
            solid_hessian_dot(l, ux, uy, uz, 0.0, 1.0, 0.0, s2[3], s2[1], t2);    // xy, yy, (zy)
            solid_hessian_dot(l, ux, uy, uz, 0.0, 0.0, 1.0, s2[4], s2[5], s2[2]); // xz, yz, zz
            (void)t0;
          }
          lcur = l;
        }
        const double R = c01.x + xs * (c01.y + xs * (c23.x + xs * c23.y));
        double f = 0.0, Rd = 0.0, hA = 0.0, hB = 0.0, hC = 0.0, qlap = 0.0;
        if (GRAD || KIN) {
          const double Rt = c01.y + xs * (2.0 * c23.x + xs * 3.0 * c23.y);
          const double sc = S.log_inc * dd;
          const double dR = Rt / sc;
          Rd = R * inv_dd;
          f = dR - (double)l * Rd;
          if (KIN || (FORCE && E.kinetic)) {
            // lap (R(d) Y_lm) = (R'' + 2 R'/d - l(l+1) R/d^2) Y_lm;  qlap = -w/4 (H planes) or -1/2 (force planes) times
            // the radial factor
            const double Rtt = 2.0 * c23.x + 6.0 * c23.y * xs;
            const double d2R = Rtt / (sc * sc) - Rt / (sc * dd);
            qlap = (FORCE ? -0.5 : -0.25 * w) * (d2R + 2.0 * dR * inv_dd - (double)(l * (l + 1)) * Rd * inv_dd);
          }
          if (HESS || FULLH) {
            // Hess phi = A u u^T Y + B (1 - u u^T) Y + B (u gS^T + gS u^T) + C Hess S, phi = (R / d^l) S_lm(dvec)
            const double Rtt = 2.0 * c23.x + 6.0 * c23.y * xs;
            const double d2R = Rtt / (sc * sc) - Rt / (sc * dd);
            hA = d2R - 2.0 * (double)l * dR * inv_dd + (double)(l * (l + 1)) * Rd * inv_dd;
            hB = f * inv_dd;
            hC = Rd * inv_dd;
          }
        }
#pragma unroll
        for (int m = 0; m < 7; m++) {
          if (m < nm) {
            const double phi = R * Y[m];
            const int oi = ro + m * mstep + (m >= wrap ? jump : 0);
            if (!TAU) op[0][oi] = phi;
            if (MODE == kEvalHLda) op[1 % NPL][oi] = wv * phi;
            if (MODE == kEvalHKinLda) op[1 % NPL][oi] = wv * phi + qlap * Y[m];
            if (GRAD) {
              const double fy = f * Y[m];
              const double ex = fy * ux + Rd * gx[m], ey = fy * uy + Rd * gy[m], ez = fy * uz + Rd * gz[m];
              if (MODE == kEvalPhiGrad || FULLH) { op[1 % NPL][oi] = ex; op[2 % NPL][oi] = ey; op[3 % NPL][oi] = ez; }
              if (FULLH) {
                const double ab = (hA - hB) * Y[m], by = hB * Y[m];
                const double ax = ab * ux + hB * gx[m], ay = ab * uy + hB * gy[m], az = ab * uz + hB * gz[m];   // u_e coefficient
                op[4 % NPL][oi] = ax * ux + hB * ux * gx[m] + by + hC * s2[0][FULLH ? m : 0];
                op[5 % NPL][oi] = ay * uy + hB * uy * gy[m] + by + hC * s2[FULLH ? 1 : 0][FULLH ? m : 0];
                op[6 % NPL][oi] = az * uz + hB * uz * gz[m] + by + hC * s2[FULLH ? 2 : 0][FULLH ? m : 0];
                op[7 % NPL][oi] = ax * uy + hB * ux * gy[m] + hC * s2[FULLH ? 3 : 0][FULLH ? m : 0];
                op[8 % NPL][oi] = ax * uz + hB * ux * gz[m] + hC * s2[FULLH ? 4 : 0][FULLH ? m : 0];
                op[9 % NPL][oi] = ay * uz + hB * uy * gz[m] + hC * s2[FULLH ? 5 : 0][FULLH ? m : 0];
              }
              if (TAU) {
                op[0][oi] = ex; op[0][oi + cstr] = ey; op[0][oi + 2 * cstr] = ez;
                op[1 % NPL][oi] = wv * ex; op[1 % NPL][oi + cstr] = wv * ey; op[1 % NPL][oi + 2 * cstr] = wv * ez;
              }
              if (MODE == kEvalHGga) op[1 % NPL][oi] = wv * phi + (wgx * ex + wgy * ey + wgz * ez);
              if (MODE == kEvalHKinGga) op[1 % NPL][oi] = wv * phi + (wgx * ex + wgy * ey + wgz * ez) + qlap * Y[m];
              if (FORCE) {
                op[1 % NPL][oi] = (HESS ? wv * phi + (wgx * ex + wgy * ey + wgz * ez) : wv * phi) + qlap * Y[m];
                op[2 % NPL][oi] = w * ex; op[3 % NPL][oi] = w * ey; op[4 % NPL][oi] = w * ez;
                if (HESS) {
                  const double gsg = gx[m] * wgx + gy[m] * wgy + gz[m] * wgz;
                  const double along = (hA - hB) * ug * Y[m] + hB * gsg;      // coefficient of u
                  const double by = hB * Y[m], bug = hB * ug;
                  op[5 % NPL][oi] = w * (along * ux + by * wgx + bug * gx[m] + hC * hx[m]);
                  op[6 % NPL][oi] = w * (along * uy + by * wgy + bug * gy[m] + hC * hy[m]);
                  op[7 % NPL][oi] = w * (along * uz + by * wgz + bug * gz[m] + hC * hz[m]);
                }
              }
            }
          }
        }
      } else {
        for (int m = 0; m < nm; m++) AIMS_EZERO(ro + m * mstep + (m >= wrap ? jump : 0))
      }
      if (AIMS_EVAL_PREFETCH) { c01 = n01; c23 = n23; }
      else if (e + 1 < n_ent) {
        const int2 en1 = s_ent[e + 1];
        const double2 *cf1 = reinterpret_cast<const double2 *>(S.spline_coef + (long long)(en1.y + k) * 4);
        if ((en1.x & 0xFF) == cur) { c01 = __ldg(cf1); c23 = __ldg(cf1 + 1); }
      }
    }
  }
#undef AIMS_EZERO
}

// copy the per-batch lists of [b0,b1) into caller arrays (aims_gpu_eval_basis outputs)
__global__ void k_export_lists(BatchLists L, DevSys S, int b0, int b1, long long *fn_ptr, int *fn_index, long long *phi_ptr,
                               const long long *api_off) {
  const int k = blockIdx.x;        // batch b0+k; block b1-b0 writes the final pointers
  const int b = b0 + k;
  if (b == b1) {
    if (threadIdx.x == 0) { fn_ptr[k] = L.fn_off[b1] - L.fn_off[b0]; phi_ptr[k] = api_off[b1] - api_off[b0]; }
    return;
  }
  const long long fo = L.fn_off[b], base = L.fn_off[b0];
  if (threadIdx.x == 0) { fn_ptr[k] = fo - base; phi_ptr[k] = api_off[b] - api_off[b0]; }
  const int nnz = L.nnz[b];
  for (int i = threadIdx.x; i < nnz; i += blockDim.x) fn_index[fo - base + i] = L.fn_index[fo + i];
}

}  // namespace aims
