// common.cuh -- shared device-side definitions of the aims_gpu CUDA path (sm_100a only).
// Product code: shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace aims {

// Static description of the system on the device (pointers into ctx-owned buffers).
struct DevSys {
  int n_atoms, n_species, n_shells, n_knots;
  const double *atom_xyz;        // [n_atoms][3]
  const int *atom_species;       // [n_atoms]
  const int *atom_fn_ptr;        // [n_atoms+1] first global function of the atom
  const int *sp_shell_ptr;       // [n_species+1]
  const double *sp_rcmax2;       // [n_species] max over shells of rcut^2
  const int *shell_l;            // [n_shells]
  const double *shell_rc2;       // [n_shells] rcut*rcut (one IEEE multiply, done on the host)
  const int *shell_spline;       // [n_shells]
  const double *spline_coef;     // [n_splines][n_knots-1][4]
  double r0, log_inc;
  // grid, structure-of-arrays
  const double *px, *py, *pz, *w;  // [n_points]
  const long long *batch_ptr;    // [n_batches+1]
  // block pattern
  const long long *row_ptr;      // [n_atoms+1]
  const int *col_atom;           // [n_blocks]
  const long long *blk_off;      // [n_blocks]
  const int *blk_ld;             // [n_blocks]
};

// Per-batch lists written by k_cull (S1a) and read by every later kernel of the same call.
struct BatchLists {
  // sized at creation from the dry run
  const long long *fn_off;       // [n_batches+1] prefix of nnz(B)
  const long long *act_off;      // [n_batches+1] prefix of n_act(B)
  const long long *ptab_off;     // [n_batches+1] prefix of n_act(B)^2
  int *nnz;                      // [n_batches]   (written by the dry run AND by every call; must agree)
  int *n_act;                    // [n_batches]
  int *fn_index;                 // [sum nnz]     global basis index, ascending per batch
  int *fn_info;                  // [sum nnz]     (slot << 16) | index of the function inside its atom's block
  int *act_atom;                 // [sum n_act]   atom id of each slot, ascending
  unsigned *act_mask;            // [sum n_act]   bit s = shell s (species-local) touches the batch
  int *act_row0;                 // [sum n_act]   first row of the slot in the batch's function list
  int *act_ld;                   // [sum n_act]   leading dimension of blocks whose column atom is this slot
  long long *ptab;               // [sum n_act^2] value offset of block (min,max) of the two slots, -1 if absent
  int *pblk;                     // [sum n_act^2] index of that block in the pattern (col_atom / blk_off numbering), -1 if absent
  int *kq;                       // [n_batches]   sum over the active atoms of their row count rounded up to even ("K'' rows")
  int *nfull;                    // [n_batches]   sum over the active atoms of ALL their functions (== nnz iff no shell is culled)
  int *error_flag;               // [1] set if a capacity was exceeded
};

constexpr int kMaxActive = 96;        // AIMS_MAX_ACTIVE_ATOMS
constexpr int kMaxCand = 1024;        // atoms passing the bounding-box test for one batch

// Internal Phi planes ("k4 layout"): rows (functions) padded with zero rows to a multiple of 8, points padded with zero
// columns to a multiple of 8; element (row, p) of a batch sits at
//     plane_offset(b) + ((p >> 2) * nnz8 + row) * 4 + (p & 3)
// so that the 8-row x 4-point operand fragment of DMMA.8x8x4 (lane = 4*row + point) is 32 consecutive doubles: one
// conflict-free LDS.64 per fragment, and any row range of one 4-point group is one contiguous segment (bulk-copyable).
// The density kernel uses the same 4-point interleave but in chunks of 16 rows ("density layout"):
//     plane_offset(b) + (((row >> 4) * (np8 >> 2) + (p >> 2)) * 16 + (row & 15)) * 4 + (p & 3),   rows padded to 16,
// so that the 16 functions of one K stage for ALL points of the batch are one contiguous segment (one bulk copy).
__host__ __device__ inline int pad8(int x) { return (x + 7) & ~7; }
__host__ __device__ inline int pad4(int x) { return (x + 3) & ~3; }

__host__ __device__ inline int round_up(int x, int m) { return (x + m - 1) / m * m; }

// ---- small PTX wrappers --------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma8x8x4(double &d0, double &d1, double a, double b) {
  // FP64 tensor-pipe MMA: D(8x8) += A(8x4) * B(4x8); SASS DMMA.8x8x4 on sm_100a.
  // lane owns A[lane>>2][lane&3], B[lane&3][lane>>2], D[lane>>2][2*(lane&3) + {0,1}]
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
// 16-byte async copy global->shared; src_bytes < 16 zero-fills the rest (0 = all zeros, nothing read)
__device__ __forceinline__ void cp_async16(unsigned dst, const void *src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async8(unsigned dst, const void *src, int src_bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }
// ---- mbarrier + 1-D bulk async copy (TMA unit; SASS UBLKCP) ---------------------------------------------------
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// global -> shared bulk copy of `bytes` (multiple of 16; both addresses 16-byte aligned), completion counted on `bar`
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// bulk prefetch of `bytes` (multiple of 16, 16-byte aligned) of global memory into L2; no completion tracking
__device__ __forceinline__ void bulk_prefetch_l2(const void *src, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(src), "r"(bytes) : "memory");
}
// the executing thread's prior cp.async operations arrive on `bar` when they complete (count not incremented)
__device__ __forceinline__ void cp_async_mbar_arrive_noinc(unsigned bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }
__device__ __forceinline__ void red_add_f64(double *addr, double v) {
  asm volatile("red.global.add.f64 [%0], %1;\n" ::"l"(addr), "d"(v) : "memory");
}

}  // namespace aims
