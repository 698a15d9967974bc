// aims_gpu.cu -- C ABI (include/aims_gpu.h) and host-side orchestration of the sm_100a kernels.
// No CPU fallback: every step of the path runs in the kernels of basis.cuh / hamiltonian.cuh / density.cuh.
#include "../../include/aims_gpu.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#if defined(AIMS_PROBE_DENSITY2) || defined(AIMS_PROBE_BALANCED_DENSITY)
#define AIMS_WITH_VARIANTS 1        // see the note at density2.cuh below; defined before basis.cuh, whose k_cull serves the variants too
#endif
#include "basis.cuh"
#include "bloch.cuh"
#include "common.cuh"
#include "density.cuh"
// The product library contains the product only.  The two measured-and-rejected density variants (density2.cuh, density_b.cuh;
// profiles/r02_kernel_experiments.md), every table, context field and launch branch that serves them, and the DMMA
// operand-pattern probes are compiled ONLY into probe builds (build.py --define AIMS_PROBE_DENSITY2=1 / AIMS_PROBE_BALANCED_DENSITY=1 /
// AIMS_PROBE_DMMA=1 --tag ...), which report their switches through aims_gpu_build_flags().
#ifdef AIMS_WITH_VARIANTS
#include "density2.cuh"
#include "density_b.cuh"
#endif
#include "forces.cuh"
#include "hessian.cuh"
#include "partition.cuh"
#include "hamiltonian.cuh"

using namespace aims;

static_assert(kMaxActive == AIMS_MAX_ACTIVE_ATOMS, "header and kernels disagree");

struct aims_gpu_ctx {
  int device = 0;
  int sm_count = 148;
  size_t smem_optin = 0;       // largest opt-in dynamic shared memory per CTA
  cudaStream_t stream = nullptr;
  std::string err;
  int64_t launches = 0;
  std::vector<void *> owned;  // device allocations to free

  DevSys S{};
  BatchLists L{};
  int n_batches = 0;
  int64_t n_points = 0, n_values = 0;

  // host copies of the static structure (dry run)
  std::vector<long long> batch_ptr, fn_off, act_off, ptab_off, pad_off, pad16_off, dpad_off, api_off, tile_off, item_off;
  std::vector<int> nnz, n_act;
  std::vector<double> h_atom_xyz;                                // host copy of the atom positions (cell lists)
  int *d_part = nullptr;                                         // flag word + cell list of aims_gpu_partition_weights (grows on demand)
  size_t part_cap = 0;
  double part_r = -1.0;                                          // r_part the cached cell list was built for (< 0: none)
  PartCells part_cells{};
  std::vector<int> h_atom_fn_ptr, h_col_atom, h_blk_ld;          // host copies of the pattern (Bloch sums)
  std::vector<long long> h_row_ptr, h_blk_off;
  int max_nnz = 0, max_act = 0, max_np = 0;
  long long *d_pad_off = nullptr, *d_pad16_off = nullptr, *d_dpad_off = nullptr, *d_api_off = nullptr;
  HTile *d_tiles = nullptr;
  DItem *d_items = nullptr;
  double flops_h_lda = 0, flops_h_gga = 0, flops_den = 0;
  bool ptab_in_smem = true, f_ptab_in_smem = true, x_ptab_in_smem = true;
  std::vector<DItem> h_items;                                  // host copy of the density work items
  std::map<std::pair<int, int>, int *> item_order;             // (bs, be) -> device permutation, heaviest item first
#ifdef AIMS_WITH_VARIANTS
  bool b_ptab_in_smem = true;
  // density_b.cuh: items of 192..224 points (update_density only; forces / Hessian keep every item in `items`)
  bool balanced_density = true;
  std::vector<long long> itemb_off, itemg_off;                 // per batch: balanced items / the other ("generic") items
  DItem *d_itemsb = nullptr, *d_itemsg = nullptr;
  std::vector<DItem> h_itemsb, h_itemsg;
  std::map<std::pair<int, int>, int *> itemb_order, itemg_order;
  // density2.cuh (bulk-copy pipeline): used when no atom of any batch is partially culled
  bool fast_density = false, d2_pblk_in_smem = true;
  std::vector<int> kq;                                         // K'' rows per batch
  int max_kq = 0;
  std::vector<long long> dq_off, item2_off;
  long long *d_dq_off = nullptr;
  DItem *d_items2 = nullptr;
  std::vector<DItem> h_items2;
  std::map<std::pair<int, int>, int *> item2_order;
  long long *d_offU = nullptr, *d_offL = nullptr;              // full-storage offsets of every pattern block
  int *d_blk_row = nullptr;
  long long full_doubles = 0, n_blocks = 0;
  double *Dfull = nullptr;                                     // full-storage copy of the density matrix (per call)
#endif

  // aims_gpu_bloch_fold: contribution lists per (cell atom, cell atom) tile, cached for the last atom_home seen
  std::vector<int> bloch_home;
  std::vector<double> bloch_T_host;
  int bloch_n_home = 0;
  BlochContrib *d_bloch_contrib = nullptr;
  int *d_bloch_tile_ptr = nullptr;
  double *d_bloch_T = nullptr;

  double *ws = nullptr;      // Phi-plane workspace
  double *probe_out = nullptr;
  bool deterministic = false;                                   // aims_gpu_set_deterministic: ordered scatter into H
  unsigned *det_counters = nullptr;                             // [2] ticket / done counters of the ordered scatter
  long long *d_tile_off = nullptr;
  long long ws_doubles = 0;

  // optional per-kernel timing (CUDA events on the context stream around every launch)
  bool timing = false;
  struct Span { cudaEvent_t e0, e1; int kind; };
  std::vector<Span> spans;       // recorded since the last read
  std::vector<Span> pool;        // reusable events
};

enum { kKindCull = 0, kKindEval = 1, kKindHam = 2, kKindDen = 3, kKindOther = 4, kKindForce = 5, kNumKinds = 6 };

namespace {

#define CU_TRY(ctx, call)                                                                          \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                             \
      return (e_ == cudaErrorMemoryAllocation) ? AIMS_ERR_NOMEM : AIMS_ERR_CUDA;                   \
    }                                                                                              \
  } while (0)

template <class T>
int dev_alloc(aims_gpu_ctx *c, T **p, size_t n) {
  void *q = nullptr;
  CU_TRY(c, cudaMalloc(&q, std::max<size_t>(n, 1) * sizeof(T)));
  c->owned.push_back(q);
  *p = static_cast<T *>(q);
  return AIMS_OK;
}
template <class T>
int dev_upload(aims_gpu_ctx *c, T **p, const T *h, size_t n) {
  int rc = dev_alloc(c, p, n);
  if (rc) return rc;
  if (n) CU_TRY(c, cudaMemcpyAsync(*p, h, n * sizeof(T), cudaMemcpyHostToDevice, c->stream));
  return AIMS_OK;
}

int fail(aims_gpu_ctx *c, int code, const char *msg) {
  if (c) c->err = msg;
  return code;
}

// asynchronous faults and capacity overflows reported by the kernels
int check_async(aims_gpu_ctx *c) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { c->err = std::string("kernel launch: ") + cudaGetErrorString(e); return AIMS_ERR_CUDA; }
  return AIMS_OK;
}

// Brackets one kernel launch with events when timing is on; always counts the launch.
struct TimedLaunch {
  aims_gpu_ctx *c;
  aims_gpu_ctx::Span sp{};
  bool on;
  TimedLaunch(aims_gpu_ctx *ctx, int kind) : c(ctx), on(ctx->timing) {
    c->launches++;
    if (!on) return;
    if (!c->pool.empty()) { sp = c->pool.back(); c->pool.pop_back(); }
    else if (cudaEventCreate(&sp.e0) != cudaSuccess || cudaEventCreate(&sp.e1) != cudaSuccess) { on = false; return; }
    sp.kind = kind;
    cudaEventRecord(sp.e0, c->stream);
  }
  ~TimedLaunch() {
    if (!on) return;
    cudaEventRecord(sp.e1, c->stream);
    c->spans.push_back(sp);
  }
};

__global__ void k_fp64_peak(double *out, int iters, double a, double b) {
  double c0[16], c1[16];
#pragma unroll
  for (int i = 0; i < 16; i++) { c0[i] = threadIdx.x * 1e-9 + i; c1[i] = i; }
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) dmma8x8x4(c0[i], c1[i], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += c0[i] + c1[i];
  if (s == 12345.678) out[0] = s;
}

#ifdef AIMS_PROBE_DMMA
// DMMA operand-pattern probe (aims_gpu_dmma_probe): one warp works on a 32x32 accumulator block, 16 DMMAs per step.
//   V = 1: operands stay in registers (4x4 outer product);  V = 2: the 8 fragments of a step are loaded from shared memory,
//   then its 16 DMMAs are issued ("load-then-compute");  V = 3: the loads of step t+1 are issued before the DMMAs of step t.
template <int V>
__global__ void __launch_bounds__(512, 1) k_dmma_probe(double *out, int iters, double a0, double b0) {
  __shared__ double sm[4096];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < 4096; i += blockDim.x) sm[i] = 1e-9 * i;
  __syncthreads();
  double acc[4][4][2];
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int c = 0; c < 4; c++) { acc[a][c][0] = a + lane; acc[a][c][1] = c; }
  double fa[4], fb[4];
#pragma unroll
  for (int a = 0; a < 4; a++) { fa[a] = a0 + a * 1e-3; fb[a] = b0 + a * 1e-4; }
  const double *tA = sm + lane + (warp & 3) * 512, *tB = sm + 2048 + lane + (warp & 3) * 512;
  if (V == 1) {
    for (int it = 0; it < iters; it++) {
#pragma unroll
      for (int a = 0; a < 4; a++)
#pragma unroll
        for (int c = 0; c < 4; c++) dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
    }
  } else if (V == 2) {
#pragma unroll 1
    for (int it = 0; it < iters; it++) {
      const int o = (it & 3) * 128;
#pragma unroll
      for (int a = 0; a < 4; a++) fa[a] = tA[o + a * 32];
#pragma unroll
      for (int c = 0; c < 4; c++) fb[c] = tB[o + c * 32];
#pragma unroll
      for (int a = 0; a < 4; a++)
#pragma unroll
        for (int c = 0; c < 4; c++) dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
    }
  } else {
    double na[4], nb[4];
#pragma unroll
    for (int a = 0; a < 4; a++) { fa[a] = tA[a * 32]; fb[a] = tB[a * 32]; }
#pragma unroll 1
    for (int it = 0; it < iters; it += 2) {
      const int o = ((it + 1) & 3) * 128, o2 = ((it + 2) & 3) * 128;
#pragma unroll
      for (int a = 0; a < 4; a++) { na[a] = tA[o + a * 32]; nb[a] = tB[o + a * 32]; }
#pragma unroll
      for (int a = 0; a < 4; a++)
#pragma unroll
        for (int c = 0; c < 4; c++) dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
#pragma unroll
      for (int a = 0; a < 4; a++) { fa[a] = tA[o2 + a * 32]; fb[a] = tB[o2 + a * 32]; }
#pragma unroll
      for (int a = 0; a < 4; a++)
#pragma unroll
        for (int c = 0; c < 4; c++) dmma8x8x4(acc[a][c][0], acc[a][c][1], na[a], nb[c]);
    }
  }
  double s = 0;
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int c = 0; c < 4; c++) s += acc[a][c][0] + acc[a][c][1];
  if (s == 12345.678) out[0] = s;
}

// Second operand-pattern probe: a (WA x WB) accumulator block per warp, WA*WB DMMAs per step.
//   INPLACE = true : the K-step body of d_mma_kloop_t / b_mma_kloop_t -- a fragment is reloaded in place (same register) as soon
//                    as the row of DMMAs that used it has been issued;
//   INPLACE = false: the fragments of step t+1 are loaded into a second register set before the DMMAs of step t.
template <int WA, int WB, bool INPLACE>
__global__ void __launch_bounds__(640) k_dmma_probe2(double *out, int iters, double a0) {
  __shared__ double sm[4096];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < 4096; i += blockDim.x) sm[i] = 1e-9 * i + a0;
  __syncthreads();
  double acc[WA][WB][2];
#pragma unroll
  for (int a = 0; a < WA; a++)
#pragma unroll
    for (int c = 0; c < WB; c++) { acc[a][c][0] = a + lane; acc[a][c][1] = c; }
  const double *tA = sm + lane + (warp & 1) * 1024, *tB = sm + 2048 + lane + (warp & 1) * 1024;
  double fa[WA], fb[WB];
#pragma unroll
  for (int a = 0; a < WA; a++) fa[a] = tA[a * 32];
#pragma unroll
  for (int c = 0; c < WB; c++) fb[c] = tB[c * 32];
  if (INPLACE) {
#pragma unroll 1
    for (int it = 0; it < iters; it++) {
      const double *a1 = tA + ((it + 1) & 3) * 256, *b1 = tB + ((it + 1) & 3) * 256;
#pragma unroll
      for (int a = 0; a < WA; a++) {
#pragma unroll
        for (int c = 0; c < WB; c++) {
          dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
          if (a == WA - 1) fb[c] = b1[c * 32];
        }
        fa[a] = a1[a * 32];
      }
    }
  } else {
    double na[WA], nb[WB];
#pragma unroll 1
    for (int it = 0; it < iters; it += 2) {
      const double *a1 = tA + ((it + 1) & 3) * 256, *b1 = tB + ((it + 1) & 3) * 256;
      const double *a2 = tA + ((it + 2) & 3) * 256, *b2 = tB + ((it + 2) & 3) * 256;
#pragma unroll
      for (int a = 0; a < WA; a++) na[a] = a1[a * 32];
#pragma unroll
      for (int c = 0; c < WB; c++) nb[c] = b1[c * 32];
#pragma unroll
      for (int a = 0; a < WA; a++)
#pragma unroll
        for (int c = 0; c < WB; c++) dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
#pragma unroll
      for (int a = 0; a < WA; a++) fa[a] = a2[a * 32];
#pragma unroll
      for (int c = 0; c < WB; c++) fb[c] = b2[c * 32];
#pragma unroll
      for (int a = 0; a < WA; a++)
#pragma unroll
        for (int c = 0; c < WB; c++) dmma8x8x4(acc[a][c][0], acc[a][c][1], na[a], nb[c]);
    }
  }
  double s = 0;
#pragma unroll
  for (int a = 0; a < WA; a++)
#pragma unroll
    for (int c = 0; c < WB; c++) s += acc[a][c][0] + acc[a][c][1];
  if (s == 12345.678) out[0] = s;
}

// Third probe: the (4 x 3) in-place K step inside the CONTROL FLOW of the kernels -- trip counts that come from global memory (so the
// compiler cannot prove them warp-uniform: vector-register loop counters, predicated branches, WARPSYNC before the DMMAs of every
// basic block), a stage loop around a step loop, and the "last step of a stage" branch that redirects the reload pointers.
//   UNROLL = false: one step per iteration of the inner loop, as d_mma_kloop_t;  true: the four steps of a stage as one block.
template <bool UNROLL>
__global__ void __launch_bounds__(640) k_dmma_probe3(double *out, const int *cnt, double a0) {
  __shared__ double sm[4096];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < 4096; i += blockDim.x) sm[i] = 1e-9 * i + a0;
  __syncthreads();
  const int nkc = cnt[0], nnz8 = cnt[1];                 // run-time values from global memory, like L.nnz[b]
  double acc[4][3][2];
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int c = 0; c < 3; c++) { acc[a][c][0] = a + lane; acc[a][c][1] = c; }
  const double *sAl = sm + lane + (warp & 1) * 1024, *sBl = sm + 2048 + lane + (warp & 1) * 1024;
  const double *tA = sAl, *tB = sBl;
  double fa[4], fb[3];
#pragma unroll
  for (int a = 0; a < 4; a++) fa[a] = tA[a * 32];
#pragma unroll
  for (int c = 0; c < 3; c++) fb[c] = tB[c * 32];
  int step = 0;
  auto one_step = [&](const double *a1, const double *b1) {
#pragma unroll
    for (int a = 0; a < 4; a++) {
#pragma unroll
      for (int c = 0; c < 3; c++) {
        dmma8x8x4(acc[a][c][0], acc[a][c][1], fa[a], fb[c]);
        if (a == 3) fb[c] = b1[c * 32];
      }
      fa[a] = a1[a * 32];
    }
  };
#pragma unroll 1
  for (int kc = 0; kc < nkc; kc++) {
    const int nk4 = min(16, nnz8 - kc * 16) >> 2;
    const bool more = kc + 1 < nkc;
    if (UNROLL && nk4 == 4) {
      one_step(tA + 128, tB + 128);
      one_step(tA + 256, tB + 256);
      one_step(tA + 384, tB + 384);
      const double *a1 = more ? sAl + ((step + 1) & 1) * 512 : tA, *b1 = more ? sBl + ((step + 1) & 1) * 512 : tB;
      one_step(a1, b1);
      tA = a1; tB = b1;
    } else {
#pragma unroll 1
      for (int t = 0; t < nk4; t++) {
        const bool last = t + 1 == nk4;
        const double *a1 = tA + (t + 1) * 128, *b1 = tB + (t + 1) * 128;
        if (last) { a1 = more ? sAl + ((step + 1) & 1) * 512 : tA; b1 = more ? sBl + ((step + 1) & 1) * 512 : tB; }
        one_step(a1, b1);
        if (last) { tA = a1; tB = b1; }
      }
    }
    step++;
  }
  double s = 0;
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int c = 0; c < 3; c++) s += acc[a][c][0] + acc[a][c][1];
  if (s == 12345.678) out[0] = s;
}

#endif  // AIMS_PROBE_DMMA

bool range_ok(const aims_gpu_ctx *c, int b0, int b1) { return c && b0 >= 0 && b1 >= b0 && b1 <= c->n_batches; }

// Every extern "C" entry runs its body through this: no C++ exception (std::bad_alloc of the host-side tables and
// strings, or anything else) crosses the C boundary -- include/aims_gpu.h promises status codes only.
template <class F>
int guarded(aims_gpu_ctx *c, F &&body) noexcept {
  try {
    return body();
  } catch (const std::bad_alloc &) {
    try { if (c) c->err = "out of host memory"; } catch (...) {}
    return AIMS_ERR_NOMEM;
  } catch (...) {
    try { if (c) c->err = "unexpected C++ exception"; } catch (...) {}
    return AIMS_ERR_INVALID_ARG;
  }
}

// Opt every kernel with dynamic shared memory in to the device maximum, ONCE per device and process.  The attribute is
// per function and device, not per context: sizing it from one context's max nnz(B) would shrink it under another,
// larger context that is still alive.
template <class K>
cudaError_t smem_optin_max(K kernel, size_t optin) {
  cudaFuncAttributes fa;
  cudaError_t e = cudaFuncGetAttributes(&fa, kernel);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(optin - fa.sharedSizeBytes));
}
constexpr size_t kStaticSmemMargin = 4096;   // >= the static shared memory of any kernel here (k_eval: 2.8 KB)

cudaError_t smem_optin_all(int device, size_t optin) {
  static std::mutex mu;
  static bool done[64] = {};
  std::lock_guard<std::mutex> lock(mu);
  if (device >= 0 && device < 64 && done[device]) return cudaSuccess;
  cudaError_t e;
#define AIMS_OPTIN(k) if ((e = smem_optin_max(k, optin)) != cudaSuccess) return e;
  AIMS_OPTIN(k_hamiltonian<false>) AIMS_OPTIN(k_hamiltonian<true>)
  AIMS_OPTIN(k_density<false>) AIMS_OPTIN(k_density<true>)
#ifdef AIMS_WITH_VARIANTS
  AIMS_OPTIN(k_density2<false>) AIMS_OPTIN(k_density2<true>)
  AIMS_OPTIN(k_density_b<false>) AIMS_OPTIN(k_density_b<true>)
  AIMS_OPTIN((k_eval<kEvalPhi, kLayD2>)) AIMS_OPTIN((k_eval<kEvalPhiGrad, kLayD2>))
#endif
  AIMS_OPTIN(k_density_hessian)
  AIMS_OPTIN((k_forces<false, false>)) AIMS_OPTIN((k_forces<true, false>))
  AIMS_OPTIN((k_forces<false, true>)) AIMS_OPTIN((k_forces<true, true>))
#define AIMS_OPTIN_EV(M, LY) AIMS_OPTIN((k_eval<M, LY>))
  AIMS_OPTIN_EV(kEvalPhi, kLayApi) AIMS_OPTIN_EV(kEvalPhiGrad, kLayApi) AIMS_OPTIN_EV(kEvalHLda, kLayH)
  AIMS_OPTIN_EV(kEvalHGga, kLayH) AIMS_OPTIN_EV(kEvalHKinLda, kLayH) AIMS_OPTIN_EV(kEvalHKinGga, kLayH)
  AIMS_OPTIN_EV(kEvalTau, kLayH) AIMS_OPTIN_EV(kEvalHess, kLayD) AIMS_OPTIN_EV(kEvalPhi, kLayD)
  AIMS_OPTIN_EV(kEvalPhiGrad, kLayD) AIMS_OPTIN_EV(kEvalForceLda, kLayD) AIMS_OPTIN_EV(kEvalForceGga, kLayD)
#undef AIMS_OPTIN_EV
#undef AIMS_OPTIN
  if (device >= 0 && device < 64) done[device] = true;
  return cudaSuccess;
}

}  // namespace

extern "C" {

const char *aims_gpu_last_error(const aims_gpu_ctx *ctx) { return ctx ? ctx->err.c_str() : ""; }
int64_t aims_gpu_launch_count(const aims_gpu_ctx *ctx) { return ctx ? ctx->launches : 0; }

int aims_gpu_destroy(aims_gpu_ctx *ctx) {
  if (!ctx) return AIMS_ERR_INVALID_ARG;
  cudaSetDevice(ctx->device);
  cudaError_t e = cudaStreamSynchronize(ctx->stream);
  for (void *p : ctx->owned) cudaFree(p);
  for (auto &sp : ctx->spans) { cudaEventDestroy(sp.e0); cudaEventDestroy(sp.e1); }
  for (auto &sp : ctx->pool) { cudaEventDestroy(sp.e0); cudaEventDestroy(sp.e1); }
  delete ctx;
  return e == cudaSuccess ? AIMS_OK : AIMS_ERR_CUDA;
}

static int impl_create(aims_gpu_ctx **out, const aims_basis_desc *B, const aims_grid_desc *G, const aims_bsr_desc *P,
                    int device, void *cuda_stream, int64_t workspace_bytes) {
  if (!out) return AIMS_ERR_INVALID_ARG;
  *out = nullptr;
  if (!B || !G || !P) return AIMS_ERR_INVALID_ARG;
  if (B->n_atoms < 0 || B->n_species <= 0 || B->n_shells <= 0 || B->n_knots < 2 || G->n_points < 0 || G->n_batches < 0 ||
      P->n_block_rows != B->n_atoms || !B->atom_xyz || !B->atom_species || !B->species_shell_ptr || !B->shell_l ||
      !B->shell_rcut || !B->shell_spline || !B->spline_coef || !G->batch_ptr || (G->n_points && (!G->xyz || !G->w)) ||
      !P->row_ptr || !P->col_atom || !P->blk_off || !P->blk_ld || !(B->r0 > 0) || !(B->log_inc > 0))
    return AIMS_ERR_INVALID_ARG;
  aims_gpu_ctx *c = new (std::nothrow) aims_gpu_ctx;
  if (!c) return AIMS_ERR_NOMEM;
  *out = c;  // returned even on failure so that the caller can read last_error, then destroy
  c->device = device;
  c->stream = static_cast<cudaStream_t>(cuda_stream);
  CU_TRY(c, cudaSetDevice(device));
  cudaDeviceProp prop;
  CU_TRY(c, cudaGetDeviceProperties(&prop, device));
  if (prop.major != 10) return fail(c, AIMS_ERR_UNSUPPORTED, "this library is built for sm_100a (B200) only");
  c->sm_count = prop.multiProcessorCount;
  c->smem_optin = (size_t)prop.sharedMemPerBlockOptin;

  // ---- validate and derive host-side tables
  const int na = B->n_atoms, nsp = B->n_species, nsh = B->n_shells;
  for (int s = 0; s < nsh; s++) {
    if (B->shell_l[s] < 0 || B->shell_l[s] > AIMS_MAX_L) return fail(c, AIMS_ERR_UNSUPPORTED, "shell_l outside 0..3");
    if (B->shell_spline[s] < 0 || B->shell_spline[s] >= B->n_splines) return fail(c, AIMS_ERR_INVALID_ARG, "shell_spline out of range");
  }
  std::vector<int> sp_nfn(nsp, 0);
  std::vector<double> sp_rcmax2(nsp, 0.0), shell_rc2(nsh);
  for (int s = 0; s < nsh; s++) shell_rc2[s] = B->shell_rcut[s] * B->shell_rcut[s];
  for (int sp = 0; sp < nsp; sp++) {
    const int s0 = B->species_shell_ptr[sp], s1 = B->species_shell_ptr[sp + 1];
    if (s0 < 0 || s1 < s0 || s1 > nsh) return fail(c, AIMS_ERR_INVALID_ARG, "species_shell_ptr not ascending");
    if (s1 - s0 > AIMS_MAX_SHELLS_PER_SPECIES) return fail(c, AIMS_ERR_UNSUPPORTED, "more than 32 shells per species");
    for (int s = s0; s < s1; s++) { sp_nfn[sp] += 2 * B->shell_l[s] + 1; sp_rcmax2[sp] = std::max(sp_rcmax2[sp], shell_rc2[s]); }
  }
  std::vector<int> atom_fn_ptr(na + 1, 0);
  for (int a = 0; a < na; a++) {
    const int sp = B->atom_species[a];
    if (sp < 0 || sp >= nsp) return fail(c, AIMS_ERR_INVALID_ARG, "atom_species out of range");
    atom_fn_ptr[a + 1] = atom_fn_ptr[a] + sp_nfn[sp];
  }
  const long long n_blocks = P->row_ptr[na];
  for (int a = 0; a < na; a++) {
    if (P->row_ptr[a + 1] <= P->row_ptr[a] || P->col_atom[P->row_ptr[a]] != a)
      return fail(c, AIMS_ERR_INVALID_ARG, "every block row must start with its diagonal block");
    for (long long q = P->row_ptr[a]; q < P->row_ptr[a + 1]; q++) {
      const int cb = P->col_atom[q];
      if (cb < a || cb >= na || (q > P->row_ptr[a] && cb <= P->col_atom[q - 1]))
        return fail(c, AIMS_ERR_INVALID_ARG, "col_atom must be ascending and >= row");
      if ((P->blk_off[q] & 1) || (P->blk_ld[q] & 1) || P->blk_ld[q] < sp_nfn[B->atom_species[cb]] ||
          P->blk_ld[q] != P->blk_ld[P->row_ptr[cb]] ||
          P->blk_off[q] + (long long)sp_nfn[B->atom_species[a]] * P->blk_ld[q] > P->n_values)
        return fail(c, AIMS_ERR_INVALID_ARG, "blk_off/blk_ld must be even, consistent per column atom and inside n_values");
    }
  }
  c->h_atom_fn_ptr = atom_fn_ptr;
  c->h_atom_xyz.assign(B->atom_xyz, B->atom_xyz + 3 * (size_t)na);
  c->h_row_ptr.assign(P->row_ptr, P->row_ptr + na + 1);
  c->h_col_atom.assign(P->col_atom, P->col_atom + n_blocks);
  c->h_blk_off.assign(P->blk_off, P->blk_off + n_blocks);
  c->h_blk_ld.assign(P->blk_ld, P->blk_ld + n_blocks);
  c->n_batches = G->n_batches;
  c->n_points = G->n_points;
  c->n_values = P->n_values;
  c->batch_ptr.assign(G->batch_ptr, G->batch_ptr + G->n_batches + 1);
  if (c->batch_ptr[0] != 0 || c->batch_ptr[G->n_batches] != G->n_points) return fail(c, AIMS_ERR_INVALID_ARG, "batch_ptr must span [0, n_points]");
  for (int b = 0; b < G->n_batches; b++) {
    const long long n = c->batch_ptr[b + 1] - c->batch_ptr[b];
    if (n < 0 || n > G->max_batch_points) return fail(c, AIMS_ERR_INVALID_ARG, "batch_ptr not ascending or batch larger than max_batch_points");
    c->max_np = std::max<int>(c->max_np, (int)n);
  }

  // ---- upload (points as structure-of-arrays)
  DevSys &S = c->S;
  S.n_atoms = na; S.n_species = nsp; S.n_shells = nsh; S.n_knots = B->n_knots;
  S.r0 = B->r0; S.log_inc = B->log_inc;
  int rc;
#define UP(field, T, hostptr, n)                                           \
  { T *d_; rc = dev_upload<T>(c, &d_, hostptr, (size_t)(n)); if (rc) return rc; field = d_; }
  UP(S.atom_xyz, double, B->atom_xyz, 3 * (size_t)na)
  UP(S.atom_species, int, B->atom_species, na)
  UP(S.atom_fn_ptr, int, atom_fn_ptr.data(), na + 1)
  UP(S.sp_shell_ptr, int, B->species_shell_ptr, nsp + 1)
  UP(S.sp_rcmax2, double, sp_rcmax2.data(), nsp)
  UP(S.shell_l, int, B->shell_l, nsh)
  UP(S.shell_rc2, double, shell_rc2.data(), nsh)
  UP(S.shell_spline, int, B->shell_spline, nsh)
  UP(S.spline_coef, double, B->spline_coef, (size_t)B->n_splines * (B->n_knots - 1) * 4)
  {
    const size_t n = (size_t)G->n_points;
    std::vector<double> soa(3 * n);
    for (size_t p = 0; p < n; p++) { soa[p] = G->xyz[3 * p]; soa[n + p] = G->xyz[3 * p + 1]; soa[2 * n + p] = G->xyz[3 * p + 2]; }
    double *d;
    rc = dev_upload<double>(c, &d, soa.data(), 3 * n);
    if (rc) return rc;
    CU_TRY(c, cudaStreamSynchronize(c->stream));  // soa goes out of scope
    S.px = d; S.py = d + n; S.pz = d + 2 * n;
  }
  UP(S.w, double, G->w, G->n_points)
  UP(S.batch_ptr, long long, c->batch_ptr.data(), G->n_batches + 1)
  {
    std::vector<long long> rp(P->row_ptr, P->row_ptr + na + 1), bo(P->blk_off, P->blk_off + n_blocks);
    UP(S.row_ptr, long long, rp.data(), na + 1)
    UP(S.blk_off, long long, bo.data(), n_blocks)
    CU_TRY(c, cudaStreamSynchronize(c->stream));
  }
  UP(S.col_atom, int, P->col_atom, n_blocks)
  UP(S.blk_ld, int, P->blk_ld, n_blocks)
#undef UP

  // ---- dry run of the culling: sizes of every per-batch list
  const int nb = c->n_batches;
  BatchLists &L = c->L;
  if ((rc = dev_alloc(c, &L.nnz, nb))) return rc;
  if ((rc = dev_alloc(c, &L.n_act, nb))) return rc;
#ifdef AIMS_WITH_VARIANTS
  if ((rc = dev_alloc(c, &L.kq, nb))) return rc;
  if ((rc = dev_alloc(c, &L.nfull, nb))) return rc;
#endif
  if ((rc = dev_alloc(c, &L.error_flag, 1))) return rc;
  CU_TRY(c, cudaMemsetAsync(L.error_flag, 0, sizeof(int), c->stream));
  if (nb) {
    { TimedLaunch t(c, kKindCull); k_cull<<<nb, 256, 0, c->stream>>>(S, L, 0, 1); }
    if ((rc = check_async(c))) return rc;
  }
  c->nnz.resize(nb); c->n_act.resize(nb);
  int flag = 0;
#ifdef AIMS_WITH_VARIANTS
  c->kq.resize(nb);
  std::vector<int> nfull(nb);
  CU_TRY(c, cudaMemcpyAsync(c->kq.data(), L.kq, nb * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  CU_TRY(c, cudaMemcpyAsync(nfull.data(), L.nfull, nb * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
#endif
  CU_TRY(c, cudaMemcpyAsync(c->nnz.data(), L.nnz, nb * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  CU_TRY(c, cudaMemcpyAsync(c->n_act.data(), L.n_act, nb * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  CU_TRY(c, cudaMemcpyAsync(&flag, L.error_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  CU_TRY(c, cudaStreamSynchronize(c->stream));
  if (flag == 1) return fail(c, AIMS_ERR_UNSUPPORTED, "more than 1024 atoms pass the bounding-box test of one batch");
  if (flag == 2) return fail(c, AIMS_ERR_UNSUPPORTED, "more than AIMS_MAX_ACTIVE_ATOMS atoms touch one batch");

  c->fn_off.assign(nb + 1, 0); c->act_off.assign(nb + 1, 0); c->ptab_off.assign(nb + 1, 0);
  c->pad_off.assign(nb + 1, 0); c->pad16_off.assign(nb + 1, 0); c->dpad_off.assign(nb + 1, 0); c->api_off.assign(nb + 1, 0); c->tile_off.assign(nb + 1, 0); c->item_off.assign(nb + 1, 0);
  std::vector<HTile> tiles;
  std::vector<DItem> items;
#ifdef AIMS_WITH_VARIANTS
  std::vector<DItem> items2, itemsb, itemsg;
  c->dq_off.assign(nb + 1, 0); c->item2_off.assign(nb + 1, 0);
  c->itemb_off.assign(nb + 1, 0); c->itemg_off.assign(nb + 1, 0);
#ifndef AIMS_PROBE_BALANCED_DENSITY
  c->balanced_density = false;       // density_b.cuh is a measured-and-rejected variant (profiles/r02_kernel_experiments.md): probe builds only
#endif
#ifdef AIMS_PROBE_DENSITY2
  c->fast_density = true;            // probe build only: the bulk-copy / two-CTA density pipeline (profiles/r02_kernel_experiments.md)
#else
  c->fast_density = false;
#endif
#endif  // AIMS_WITH_VARIANTS
  for (int b = 0; b < nb; b++) {
#ifdef AIMS_WITH_VARIANTS
    if (nfull[b] != c->nnz[b]) c->fast_density = false;          // an atom lost some of its shells: density.cuh handles that
    c->max_kq = std::max(c->max_kq, c->kq[b]);
    {
      const int np_ = (int)(c->batch_ptr[b + 1] - c->batch_ptr[b]), np8_ = pad8(np_);
      c->dq_off[b + 1] = c->dq_off[b] + (long long)round_up(c->kq[b], 16) * np8_;
      if (c->nnz[b] > 0 && np_ > 0) {
        const int nsub = np8_ >> 3, nit = (np8_ + kD2MaxPts - 1) / kD2MaxPts;
        for (int q = 0; q < nit; q++) {
          const int s0 = (int)((long long)q * nsub / nit), s1 = (int)((long long)(q + 1) * nsub / nit);
          if (s1 > s0) items2.push_back(DItem{b, s0 * 8, (s1 - s0) * 8, 0});
        }
      }
      c->item2_off[b + 1] = (long long)items2.size();
    }
#endif
    const int nz = c->nnz[b], nact = c->n_act[b];
    const int np = (int)(c->batch_ptr[b + 1] - c->batch_ptr[b]);
    const int nz8 = pad8(nz), np8 = pad8(np);
    c->max_nnz = std::max(c->max_nnz, nz);
    c->max_act = std::max(c->max_act, nact);
    c->fn_off[b + 1] = c->fn_off[b] + nz;
    c->act_off[b + 1] = c->act_off[b] + nact;
    c->ptab_off[b + 1] = c->ptab_off[b] + (long long)nact * nact;
    c->pad_off[b + 1] = c->pad_off[b] + (long long)nz8 * np8;                 // H layout
    c->pad16_off[b + 1] = c->pad16_off[b] + (long long)nz8 * round_up(np, 16);   // H layout of the LDA planes (16-point stages)
    c->dpad_off[b + 1] = c->dpad_off[b] + (long long)round_up(nz, 16) * np8;   // density layout
    c->api_off[b + 1] = c->api_off[b] + (long long)nz * np;
    // Hamiltonian tiles: I panels of kHIB blocks x J panels of kHJB blocks that contain a block (bi, bj >= bi)
    if (nz > 0 && np > 0) {
      const int nblk = blk_count(nz8 >> 3);
      for (int ti = 0; ti * kHIB < nblk; ti++)
        for (int tj = 0; tj * kHJB < nblk; tj++)
          if (std::min(tj * kHJB + kHJB, nblk) - 1 >= ti * kHIB) tiles.push_back(HTile{b, (short)ti, (short)tj});
    }
    c->tile_off[b + 1] = (long long)tiles.size();
    // density items: balanced ranges of <= kDNP points, multiples of 8
    if (nz > 0 && np > 0) {
      const int nsub = np8 >> 3, nit = (np8 + kDNP - 1) / kDNP;
      const int bal = (nsub + nit - 1) / nit;                      // sub-tiles of the largest item of a balanced split
      if (nit > 1 && bal > 16 && bal <= 20 && nsub - (nit - 1) * (kDNP >> 3) >= 6) {
        // a balanced split would give items of 5 point blocks, which occupy only 10 of the 14 MMA warps: take full
        // 224-point items and one remainder item instead
        for (int q = 0, s0 = 0; q < nit; q++) {
          const int s1 = std::min(nsub, s0 + (kDNP >> 3));
          items.push_back(DItem{b, s0 * 8, (s1 - s0) * 8, 0});
          s0 = s1;
        }
      } else {
        for (int q = 0; q < nit; q++) {
          const int s0 = (int)((long long)q * nsub / nit), s1 = (int)((long long)(q + 1) * nsub / nit);
          if (s1 > s0) items.push_back(DItem{b, s0 * 8, (s1 - s0) * 8, 0});
        }
      }
    }
#ifdef AIMS_WITH_VARIANTS
    for (size_t q = (size_t)c->item_off[b]; q < items.size(); q++)
      (c->balanced_density && b_item_ok(items[q].npt) ? itemsb : itemsg).push_back(items[q]);
    c->itemb_off[b + 1] = (long long)itemsb.size();
    c->itemg_off[b + 1] = (long long)itemsg.size();
#endif
    c->item_off[b + 1] = (long long)items.size();
    c->flops_h_lda += (double)np * nz * (nz + 1.0);
    c->flops_h_gga += 2.0 * np * (double)nz * nz;
    c->flops_den += 2.0 * np * (double)nz * nz;
  }
  if (c->max_nnz >= 65536) return fail(c, AIMS_ERR_UNSUPPORTED, "nnz(B) >= 65536");
  {
    long long *d;
#define UPL(vec, field) if ((rc = dev_upload<long long>(c, &d, vec.data(), vec.size()))) return rc; field = d;
    UPL(c->fn_off, L.fn_off) UPL(c->act_off, L.act_off) UPL(c->ptab_off, L.ptab_off)
    UPL(c->pad_off, c->d_pad_off) UPL(c->pad16_off, c->d_pad16_off) UPL(c->dpad_off, c->d_dpad_off) UPL(c->api_off, c->d_api_off)
#undef UPL
  }
  if ((rc = dev_upload<HTile>(c, &c->d_tiles, tiles.data(), tiles.size()))) return rc;
  if ((rc = dev_upload<DItem>(c, &c->d_items, items.data(), items.size()))) return rc;
  c->h_items = items;
#ifdef AIMS_WITH_VARIANTS
  if ((rc = dev_upload<DItem>(c, &c->d_itemsb, itemsb.data(), itemsb.size()))) return rc;
  if ((rc = dev_upload<DItem>(c, &c->d_itemsg, itemsg.data(), itemsg.size()))) return rc;
  c->h_itemsb = itemsb; c->h_itemsg = itemsg;
  if ((rc = dev_upload<DItem>(c, &c->d_items2, items2.data(), items2.size()))) return rc;
  c->h_items2 = items2;
  if ((rc = dev_upload<long long>(c, &c->d_dq_off, c->dq_off.data(), c->dq_off.size()))) return rc;
  {
    // full-storage layout of a pattern matrix (density2.cuh: k_expand_matrix): U part of block (A,B), L part = block (B,A)
    std::vector<long long> offU((size_t)n_blocks), offL((size_t)n_blocks);
    std::vector<int> blk_row((size_t)n_blocks);
    long long off = 512;                                         // [0, 512): the zero page
    for (int a = 0; a < na; a++)
      for (long long q = P->row_ptr[a]; q < P->row_ptr[a + 1]; q++) {
        const int bb = P->col_atom[q];
        const long long nA = atom_fn_ptr[a + 1] - atom_fn_ptr[a], nB = atom_fn_ptr[bb + 1] - atom_fn_ptr[bb];
        blk_row[(size_t)q] = a;
        offU[(size_t)q] = off; off += nA * ((nB + 1) & ~1ll);
        offL[(size_t)q] = off; if (bb != a) off += nB * ((nA + 1) & ~1ll);
      }
    c->full_doubles = off; c->n_blocks = n_blocks;
    if ((rc = dev_upload<long long>(c, &c->d_offU, offU.data(), offU.size()))) return rc;
    if ((rc = dev_upload<long long>(c, &c->d_offL, offL.data(), offL.size()))) return rc;
    if ((rc = dev_upload<int>(c, &c->d_blk_row, blk_row.data(), blk_row.size()))) return rc;
    CU_TRY(c, cudaStreamSynchronize(c->stream));
  }
#endif
  CU_TRY(c, cudaStreamSynchronize(c->stream));
  if ((rc = dev_alloc(c, &L.fn_index, (size_t)c->fn_off[nb]))) return rc;
  if ((rc = dev_alloc(c, &L.fn_info, (size_t)c->fn_off[nb]))) return rc;
  if ((rc = dev_alloc(c, &L.act_atom, (size_t)c->act_off[nb]))) return rc;
  if ((rc = dev_alloc(c, &L.act_mask, (size_t)c->act_off[nb]))) return rc;
  if ((rc = dev_alloc(c, &L.act_row0, (size_t)c->act_off[nb]))) return rc;
  if ((rc = dev_alloc(c, &L.act_ld, (size_t)c->act_off[nb]))) return rc;
  if ((rc = dev_alloc(c, &L.ptab, (size_t)c->ptab_off[nb]))) return rc;
#ifdef AIMS_WITH_VARIANTS
  if ((rc = dev_alloc(c, &L.pblk, (size_t)c->ptab_off[nb]))) return rc;
#endif

  // ---- Phi-plane workspace: at least the largest single batch in EVERY plane layout used by a call (10 planes of the
  // density layout for the Hessian, 6 x the 16-point-padded H layout for the tau matrix), at most the requested budget
  long long want = workspace_bytes > 0 ? workspace_bytes : (24ll << 30);
  size_t free_b = 0, total_b = 0;
  CU_TRY(c, cudaMemGetInfo(&free_b, &total_b));
  want = std::min<long long>(want, (long long)(free_b * 0.8));
  long long need_min = 0;
  for (int b = 0; b < nb; b++)
    need_min = std::max({need_min, 10 * (c->dpad_off[b + 1] - c->dpad_off[b]), 6 * (c->pad16_off[b + 1] - c->pad16_off[b]),
                         2 * (c->pad_off[b + 1] - c->pad_off[b])});
  long long need_all = std::max({10 * c->dpad_off[nb], 6 * c->pad16_off[nb], 2 * c->pad_off[nb]});
#ifdef AIMS_WITH_VARIANTS
  for (int b = 0; b < nb; b++) need_min = std::max(need_min, 4 * (c->dq_off[b + 1] - c->dq_off[b]));
  need_all = std::max(need_all, 4 * c->dq_off[nb]);
#endif
  long long wsd = std::min(need_all, std::max(want / 8, need_min)) + 10 * 64;
  if (wsd * 8 > (long long)free_b) return fail(c, AIMS_ERR_NOMEM, "not enough device memory for one batch of Phi planes");
  if ((rc = dev_alloc(c, &c->ws, (size_t)wsd))) return rc;
  c->ws_doubles = wsd;
  if ((rc = dev_alloc(c, &c->det_counters, 2))) return rc;
  if ((rc = dev_upload<long long>(c, &c->d_tile_off, c->tile_off.data(), c->tile_off.size()))) return rc;

  // large dynamic shared memory: every kernel is opted in to the device maximum once per device (see smem_optin_all);
  // here only this context's own requirements are checked against it
  CU_TRY(c, smem_optin_all(device, c->smem_optin));
  const size_t lim = c->smem_optin - kStaticSmemMargin;
  const int mact = std::max(c->max_act, 1);
  c->ptab_in_smem = d_smem_bytes(c->max_nnz, mact, true) <= lim;
  if (d_smem_bytes(c->max_nnz, mact, c->ptab_in_smem) > lim)
    return fail(c, AIMS_ERR_UNSUPPORTED, "nnz(B) too large for the density kernel's shared memory");
#ifdef AIMS_WITH_VARIANTS
  c->b_ptab_in_smem = b_smem_bytes(c->max_nnz, mact, true) <= lim;
  if (b_smem_bytes(c->max_nnz, mact, c->b_ptab_in_smem) > lim)
    return fail(c, AIMS_ERR_UNSUPPORTED, "nnz(B) too large for the density kernel's shared memory");
#endif
  c->x_ptab_in_smem = x_smem_bytes(c->max_nnz, mact, true) <= lim;
  c->f_ptab_in_smem = f_smem_bytes(c->max_nnz, mact, true) <= lim;
  if (f_smem_bytes(c->max_nnz, mact, c->f_ptab_in_smem) > lim)
    return fail(c, AIMS_ERR_UNSUPPORTED, "nnz(B) too large for the force kernel's shared memory");
  if (eval_smem_bytes(c->max_nnz) > lim)
    return fail(c, AIMS_ERR_UNSUPPORTED, "nnz(B) too large for the evaluation kernel's shared memory");
#ifdef AIMS_WITH_VARIANTS
  c->d2_pblk_in_smem = d2_smem_bytes(c->max_nnz, c->max_kq, mact, true) <= lim / 2;      // two CTAs per SM
  if (d2_smem_bytes(c->max_nnz, c->max_kq, mact, c->d2_pblk_in_smem) > lim) c->fast_density = false;
  if (c->fast_density && (rc = dev_alloc(c, &c->Dfull, (size_t)c->full_doubles))) return rc;
  if (c->fast_density) CU_TRY(c, cudaMemsetAsync(c->Dfull, 0, 512 * sizeof(double), c->stream));
#endif
  CU_TRY(c, cudaStreamSynchronize(c->stream));
  return AIMS_OK;
}

static int impl_stats(aims_gpu_ctx *c, int64_t *sum_nnz, int32_t *max_nnz, int32_t *max_active_atoms, double *flops_h_lda,
                   double *flops_h_gga, double *flops_density) {
  if (!c) return AIMS_ERR_INVALID_ARG;
  if (sum_nnz) *sum_nnz = c->fn_off.empty() ? 0 : c->fn_off.back();
  if (max_nnz) *max_nnz = c->max_nnz;
  if (max_active_atoms) *max_active_atoms = c->max_act;
  if (flops_h_lda) *flops_h_lda = c->flops_h_lda;
  if (flops_h_gga) *flops_h_gga = c->flops_h_gga;
  if (flops_density) *flops_density = c->flops_den;
  return AIMS_OK;
}

static int impl_batch_nnz(aims_gpu_ctx *c, int32_t *nnz) {
  if (!c || !nnz) return AIMS_ERR_INVALID_ARG;
  std::copy(c->nnz.begin(), c->nnz.end(), nnz);
  return AIMS_OK;
}

static int impl_basis_sizes(aims_gpu_ctx *c, int32_t b0, int32_t b1, int64_t *n_index, int64_t *n_phi) {
  if (!range_ok(c, b0, b1)) return fail(c, AIMS_ERR_INVALID_ARG, "batch range outside [0, n_batches]");
  if (n_index) *n_index = c->fn_off[b1] - c->fn_off[b0];
  if (n_phi) *n_phi = c->api_off[b1] - c->api_off[b0];
  return AIMS_OK;
}

}  // extern "C"

namespace {

// S1a for batches [b0,b1): rebuilds every per-batch list on the device (part of each hot call)
int run_cull(aims_gpu_ctx *c, int b0, int b1) {
  if (b1 > b0) {
    TimedLaunch t(c, kKindCull);
    k_cull<<<b1 - b0, 256, 0, c->stream>>>(c->S, c->L, b0, 0);
  }
  return check_async(c);
}

// last batch (exclusive) of the chunk starting at bs such that nplanes planes fit the workspace
// (-1: even one batch does not fit -- cannot happen for the layouts create sized the workspace for)
int chunk_end(const aims_gpu_ctx *c, const std::vector<long long> &off, int bs, int b1, int nplanes) {
  const long long cap = (c->ws_doubles / nplanes) & ~63ll;   // plane stride: 512-byte aligned
  if (off[bs + 1] - off[bs] > cap) return -1;
  int lo = bs + 1, hi = b1;
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (off[mid] - off[bs] <= cap) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// Launch order of the density items of batches [bs, be): heaviest (largest nnz) first, so that the last CTAs of a launch
// are the cheapest ones (a CTA's cost varies by 50x over a slab).  Built once per distinct range and kept on the device.
enum { kItemsAll = 0, kItemsV2 = 1, kItemsBalanced = 2, kItemsGeneric = 3 };
int density_order(aims_gpu_ctx *c, int bs, int be, const int **out, int which = kItemsAll) {
#ifdef AIMS_WITH_VARIANTS
  const std::vector<long long> &ioff = which == kItemsV2 ? c->item2_off : which == kItemsBalanced ? c->itemb_off
                                       : which == kItemsGeneric ? c->itemg_off : c->item_off;
  const std::vector<DItem> &hitems = which == kItemsV2 ? c->h_items2 : which == kItemsBalanced ? c->h_itemsb
                                     : which == kItemsGeneric ? c->h_itemsg : c->h_items;
  std::map<std::pair<int, int>, int *> &cache = which == kItemsV2 ? c->item2_order : which == kItemsBalanced ? c->itemb_order
                                                : which == kItemsGeneric ? c->itemg_order : c->item_order;
#else
  (void)which;
  const std::vector<long long> &ioff = c->item_off;
  const std::vector<DItem> &hitems = c->h_items;
  std::map<std::pair<int, int>, int *> &cache = c->item_order;
#endif
  const long long i0 = ioff[bs], i1 = ioff[be];
  if (i1 - i0 <= 2ll * c->sm_count) { *out = nullptr; return AIMS_OK; }   // fewer items than two waves: any order
  auto key = std::make_pair(bs, be);
  auto it = cache.find(key);
  if (it != cache.end()) { *out = it->second; return AIMS_OK; }
  if (cache.size() >= 64) {
    // a caller walking over many distinct ranges: do not let the cache grow without bound
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    for (auto &kv : cache) {
      c->owned.erase(std::remove(c->owned.begin(), c->owned.end(), (void *)kv.second), c->owned.end());
      cudaFree(kv.second);
    }
    cache.clear();
  }
  std::vector<int> ord((size_t)(i1 - i0));
  for (long long i = i0; i < i1; i++) ord[(size_t)(i - i0)] = (int)(i - i0);
  std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) {
    const DItem &x = hitems[(size_t)(i0 + a)], &y = hitems[(size_t)(i0 + b)];
#ifdef AIMS_WITH_VARIANTS
    if (which == kItemsV2) return c->nnz[x.b] > c->nnz[y.b];       // the items of one batch stay neighbours: they read the same D_b pieces (L2)
#endif
    const long long cx = (long long)c->nnz[x.b] * c->nnz[x.b] * x.npt, cy = (long long)c->nnz[y.b] * c->nnz[y.b] * y.npt;
    return cx > cy;
  });
  int *d = nullptr;
  int rc = dev_upload<int>(c, &d, ord.data(), ord.size());
  if (rc) return rc;
  CU_TRY(c, cudaStreamSynchronize(c->stream));   // ord is a temporary
  cache[key] = d;
  *out = d;
  return AIMS_OK;
}

// One k_hamiltonian launch over the tiles of batches [bs, ...).  In deterministic mode (aims_gpu_set_deterministic) the
// CTAs take their tile from a ticket counter and scatter in batch order (hamiltonian.cuh: "ordered scatter").
int launch_hamiltonian(aims_gpu_ctx *c, bool syr2k, HArgs A, int bs, long long nt) {
  if (c->deterministic) {
    CU_TRY(c, cudaMemsetAsync(c->det_counters, 0, 2 * sizeof(unsigned), c->stream));
    A.det = 1; A.ticket = c->det_counters; A.done = c->det_counters + 1;
    A.tile_off = c->d_tile_off; A.tile_base = c->tile_off[bs];
  }
  TimedLaunch t(c, kKindHam);
  if (syr2k) k_hamiltonian<true><<<(unsigned)nt, kHThreads, h_smem_bytes<true>(), c->stream>>>(c->S, c->L, A);
  else k_hamiltonian<false><<<(unsigned)nt, kHThreads, h_smem_bytes<false>(), c->stream>>>(c->S, c->L, A);
  return AIMS_OK;
}

template <int MODE, int LAYOUT>
void launch_eval(aims_gpu_ctx *c, const EvalArgs &E, int bs, int be) {
  TimedLaunch t(c, kKindEval);
  k_eval<MODE, LAYOUT><<<be - bs, kEvalThreads, eval_smem_bytes(c->max_nnz), c->stream>>>(c->S, c->L, E, bs, std::max(c->max_nnz, 1));
}

}  // namespace

extern "C" {

static int impl_eval_basis(aims_gpu_ctx *c, int32_t b0, int32_t b1, int64_t *fn_ptr, int32_t *fn_index, int64_t *phi_ptr,
                        double *phi, double *dphi) {
  if (!range_ok(c, b0, b1)) return fail(c, AIMS_ERR_INVALID_ARG, "batch range outside [0, n_batches]");
  if (!fn_ptr || !fn_index || !phi_ptr || !phi) return fail(c, AIMS_ERR_INVALID_ARG, "NULL output");
  CU_TRY(c, cudaSetDevice(c->device));
  int rc = run_cull(c, b0, b1);
  if (rc) return rc;
  { TimedLaunch t(c, kKindOther);
    k_export_lists<<<b1 - b0 + 1, 128, 0, c->stream>>>(c->L, c->S, b0, b1, (long long *)fn_ptr, fn_index, (long long *)phi_ptr, c->d_api_off); }
  if (b1 > b0) {
    EvalArgs E{};
    E.plane[0] = phi; E.plane[1] = dphi;
    E.api_off = c->d_api_off; E.api_base = c->api_off[b0];
    E.n_points = c->n_points;
    if (dphi) launch_eval<kEvalPhiGrad, kLayApi>(c, E, b0, b1); else launch_eval<kEvalPhi, kLayApi>(c, E, b0, b1);
  }
  return check_async(c);
}

static int run_hamiltonian(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, int kinetic,
                           double *H_values, int accumulate) {
  if (!range_ok(c, b0, b1)) return fail(c, AIMS_ERR_INVALID_ARG, "batch range outside [0, n_batches]");
  if ((!v && c->n_points) || !H_values) return fail(c, AIMS_ERR_INVALID_ARG, "NULL v or H_values");
  CU_TRY(c, cudaSetDevice(c->device));
  if (!accumulate) CU_TRY(c, cudaMemsetAsync(H_values, 0, (size_t)c->n_values * sizeof(double), c->stream));
  int rc = run_cull(c, b0, b1);
  if (rc) return rc;
  const bool syr2k = g || kinetic;     // Q is not proportional to P: P Q^T + Q P^T
  // the LDA kernel runs 16-point stages on planes padded to a multiple of 16 points
  const std::vector<long long> &poff = syr2k ? c->pad_off : c->pad16_off;
  const long long *d_poff = syr2k ? c->d_pad_off : c->d_pad16_off;
  for (int bs = b0; bs < b1;) {
    const int be = chunk_end(c, poff, bs, b1, 2);
    if (be < 0) return fail(c, AIMS_ERR_NOMEM, "workspace too small for one batch of Phi planes");
    const long long plane = (c->ws_doubles / 2) & ~63ll;
    EvalArgs E{};
    E.plane[0] = c->ws; E.plane[1] = c->ws + plane;
    E.pad_off = d_poff; E.pad_base = poff[bs]; E.point_pad = syr2k ? 8 : 16;
    E.v = v; E.g = g; E.n_points = c->n_points;
    if (kinetic) { if (g) launch_eval<kEvalHKinGga, kLayH>(c, E, bs, be); else launch_eval<kEvalHKinLda, kLayH>(c, E, bs, be); }
    else if (g) launch_eval<kEvalHGga, kLayH>(c, E, bs, be);
    else launch_eval<kEvalHLda, kLayH>(c, E, bs, be);
    const long long nt = c->tile_off[be] - c->tile_off[bs];
    if (nt > 0) {
      HArgs A{c->d_tiles + c->tile_off[bs], E.plane[0], E.plane[1], d_poff, poff[bs], H_values, 1};
      if ((rc = launch_hamiltonian(c, syr2k, A, bs, nt))) return rc;
    }
    if ((rc = check_async(c))) return rc;
    bs = be;
  }
  return AIMS_OK;
}

static int impl_add_tau_matrix(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *xi, double *H_values) {
  if (!range_ok(c, b0, b1)) return fail(c, AIMS_ERR_INVALID_ARG, "batch range outside [0, n_batches]");
  if ((!xi && c->n_points) || !H_values) return fail(c, AIMS_ERR_INVALID_ARG, "NULL xi or H_values");
  CU_TRY(c, cudaSetDevice(c->device));
  int rc = run_cull(c, b0, b1);
  if (rc) return rc;
  for (int bs = b0; bs < b1;) {
    // two planes of 3 x the 16-padded points each: [d_x Phi | d_y Phi | d_z Phi] and w xi / 2 times it
    const int be = chunk_end(c, c->pad16_off, bs, b1, 6);
    if (be < 0) return fail(c, AIMS_ERR_NOMEM, "workspace too small for one batch of Phi planes");
    const long long third = (c->ws_doubles / 6) & ~63ll;
    EvalArgs E{};
    E.plane[0] = c->ws; E.plane[1] = c->ws + 3 * third;
    E.pad_off = c->d_pad16_off; E.pad_base = c->pad16_off[bs]; E.point_pad = 16;
    E.v = xi; E.n_points = c->n_points;
    launch_eval<kEvalTau, kLayH>(c, E, bs, be);
    const long long nt = c->tile_off[be] - c->tile_off[bs];
    if (nt > 0) {
      HArgs A{c->d_tiles + c->tile_off[bs], E.plane[0], E.plane[1], c->d_pad16_off, c->pad16_off[bs], H_values, 3};
      if ((rc = launch_hamiltonian(c, false, A, bs, nt))) return rc;
    }
    if ((rc = check_async(c))) return rc;
    bs = be;
  }
  return AIMS_OK;
}

static int impl_integrate_hamiltonian(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g,
                                   double *H_values, int accumulate) {
  return run_hamiltonian(c, b0, b1, v, g, 0, H_values, accumulate);
}

static int impl_integrate_hamiltonian_ks(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, int kinetic,
                                      double *H_values, int accumulate) {
  return run_hamiltonian(c, b0, b1, v, g, kinetic, H_values, accumulate);
}

static int impl_update_density(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *D_values, double *n, double *grad_n) {
  if (!range_ok(c, b0, b1)) return fail(c, AIMS_ERR_INVALID_ARG, "batch range outside [0, n_batches]");
  if (!D_values || (!n && c->n_points)) return fail(c, AIMS_ERR_INVALID_ARG, "NULL D_values or n");
  CU_TRY(c, cudaSetDevice(c->device));
  int rc = run_cull(c, b0, b1);
  if (rc) return rc;
  const int npl = grad_n ? 4 : 1;
#ifdef AIMS_WITH_VARIANTS
  if (c->fast_density && b1 > b0) {
    // density2.cuh: D written out in full storage once, then per chunk k_eval<., kLayD2> + k_density2
    ExpandArgs X{D_values, c->Dfull, c->d_offU, c->d_offL, c->d_blk_row, 512};
    if (c->n_blocks > 0) {
      TimedLaunch t(c, kKindOther);
      k_expand_matrix<<<(unsigned)c->n_blocks, 256, 0, c->stream>>>(c->S, X, c->n_blocks);
    }
    const int mact = std::max(c->max_act, 1);
    const size_t dsm2 = d2_smem_bytes(c->max_nnz, c->max_kq, mact, c->d2_pblk_in_smem);
    for (int bs = b0; bs < b1;) {
      const int be = chunk_end(c, c->dq_off, bs, b1, npl);
      if (be < 0) return fail(c, AIMS_ERR_NOMEM, "workspace too small for one batch of Phi planes");
      const long long plane = (c->ws_doubles / npl) & ~63ll;
      EvalArgs E{};
      for (int q = 0; q < npl; q++) E.plane[q] = c->ws + q * plane;
      if (!grad_n) E.plane[1] = c->ws;
      E.pad_off = c->d_dq_off; E.pad_base = c->dq_off[bs];
      E.n_points = c->n_points;
      if (grad_n) launch_eval<kEvalPhiGrad, kLayD2>(c, E, bs, be); else launch_eval<kEvalPhi, kLayD2>(c, E, bs, be);
      const long long ni = c->item2_off[be] - c->item2_off[bs];
      if (ni > 0) {
        D2Args A{};
        if ((rc = density_order(c, bs, be, &A.order, kItemsV2))) return rc;
        A.items = c->d_items2 + c->item2_off[bs];
        A.P = E.plane[0];
        for (int q = 0; q < 3; q++) A.G[q] = grad_n ? E.plane[q + 1] : nullptr;
        A.pad_off = c->d_dq_off; A.pad_base = c->dq_off[bs];
        A.F = c->Dfull; A.offU = c->d_offU; A.offL = c->d_offL;
        A.n = n; A.gn = grad_n; A.n_points = c->n_points; A.max_nnz_pad = c->max_nnz; A.max_kq_pad = c->max_kq;
        A.pblk_in_smem = c->d2_pblk_in_smem ? 1 : 0;
        TimedLaunch t(c, kKindDen);
        if (grad_n) k_density2<true><<<(unsigned)ni, kD2Threads, dsm2, c->stream>>>(c->S, c->L, A, mact);
        else k_density2<false><<<(unsigned)ni, kD2Threads, dsm2, c->stream>>>(c->S, c->L, A, mact);
      }
      if ((rc = check_async(c))) return rc;
      bs = be;
    }
    return AIMS_OK;
  }
#endif
  const size_t dsm = d_smem_bytes(c->max_nnz, std::max(c->max_act, 1), c->ptab_in_smem);
  for (int bs = b0; bs < b1;) {
    const int be = chunk_end(c, c->dpad_off, bs, b1, npl);
    if (be < 0) return fail(c, AIMS_ERR_NOMEM, "workspace too small for one batch of Phi planes");
    const long long plane = (c->ws_doubles / npl) & ~63ll;
    EvalArgs E{};
    for (int q = 0; q < npl; q++) E.plane[q] = c->ws + q * plane;
    if (!grad_n) E.plane[1] = c->ws;  // unused
    E.pad_off = c->d_dpad_off; E.pad_base = c->dpad_off[bs];
    E.n_points = c->n_points;
    if (grad_n) launch_eval<kEvalPhiGrad, kLayD>(c, E, bs, be); else launch_eval<kEvalPhi, kLayD>(c, E, bs, be);
#ifdef AIMS_WITH_VARIANTS
    // items of 192..224 points (all of a 200-point configuration) -> k_density_b, the others -> k_density
    const long long nib = c->itemb_off[be] - c->itemb_off[bs], nig = c->itemg_off[be] - c->itemg_off[bs];
#else
    const long long nig = c->item_off[be] - c->item_off[bs];
#endif
    DArgs A{};
    A.P = E.plane[0];
    for (int q = 0; q < 3; q++) A.G[q] = grad_n ? E.plane[q + 1] : nullptr;
    A.pad_off = c->d_dpad_off; A.pad_base = c->dpad_off[bs];
    A.D = D_values; A.n = n; A.gn = grad_n; A.n_points = c->n_points; A.max_nnz_pad = c->max_nnz;
#ifdef AIMS_WITH_VARIANTS
    if (nib > 0) {
      if ((rc = density_order(c, bs, be, &A.order, kItemsBalanced))) return rc;
      A.items = c->d_itemsb + c->itemb_off[bs];
      A.ptab_in_smem = c->b_ptab_in_smem ? 1 : 0;
      const size_t bsm = b_smem_bytes(c->max_nnz, std::max(c->max_act, 1), c->b_ptab_in_smem);
      TimedLaunch t(c, kKindDen);
      if (grad_n) k_density_b<true><<<(unsigned)nib, kBThreads, bsm, c->stream>>>(c->S, c->L, A, std::max(c->max_act, 1));
      else k_density_b<false><<<(unsigned)nib, kBThreads, bsm, c->stream>>>(c->S, c->L, A, std::max(c->max_act, 1));
    }
#endif
    if (nig > 0) {
#ifdef AIMS_WITH_VARIANTS
      if ((rc = density_order(c, bs, be, &A.order, kItemsGeneric))) return rc;
      A.items = c->d_itemsg + c->itemg_off[bs];
#else
      if ((rc = density_order(c, bs, be, &A.order))) return rc;
      A.items = c->d_items + c->item_off[bs];
#endif
      A.ptab_in_smem = c->ptab_in_smem ? 1 : 0;
      TimedLaunch t(c, kKindDen);
      if (grad_n) k_density<true><<<(unsigned)nig, kDThreads, dsm, c->stream>>>(c->S, c->L, A, std::max(c->max_act, 1));
      else k_density<false><<<(unsigned)nig, kDThreads, dsm, c->stream>>>(c->S, c->L, A, std::max(c->max_act, 1));
    }
    if ((rc = check_async(c))) return rc;
    bs = be;
  }
  return AIMS_OK;
}

static int run_forces(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, int kinetic,
                      const double *D_values, const double *Q_values, double *F, int accumulate, double *sigma = nullptr,
                      double volume = 1.0) {
  if (!range_ok(c, b0, b1)) return fail(c, AIMS_ERR_INVALID_ARG, "batch range outside [0, n_batches]");
  if ((!v && c->n_points) || !D_values || (!F && !sigma)) return fail(c, AIMS_ERR_INVALID_ARG, "NULL v, D_values or F");
  if (sigma && !(volume > 0.0)) return fail(c, AIMS_ERR_INVALID_ARG, "volume must be positive");
  CU_TRY(c, cudaSetDevice(c->device));
  if (!accumulate && F) CU_TRY(c, cudaMemsetAsync(F, 0, (size_t)c->S.n_atoms * 3 * sizeof(double), c->stream));
  if (!accumulate && sigma) CU_TRY(c, cudaMemsetAsync(sigma, 0, 9 * sizeof(double), c->stream));
  int rc = run_cull(c, b0, b1);
  if (rc) return rc;
  const int npl = g ? 8 : 5;
  const size_t fsm = f_smem_bytes(c->max_nnz, std::max(c->max_act, 1), c->f_ptab_in_smem);
  for (int bs = b0; bs < b1;) {
    const int be = chunk_end(c, c->dpad_off, bs, b1, npl);
    if (be < 0) return fail(c, AIMS_ERR_NOMEM, "workspace too small for one batch of Phi planes");
    const long long plane = (c->ws_doubles / npl) & ~63ll;
    EvalArgs E{};
    for (int q = 0; q < npl; q++) E.plane[q] = c->ws + q * plane;
    E.pad_off = c->d_dpad_off; E.pad_base = c->dpad_off[bs];
    E.v = v; E.g = g; E.n_points = c->n_points; E.kinetic = kinetic ? 1 : 0;
    if (g) launch_eval<kEvalForceGga, kLayD>(c, E, bs, be); else launch_eval<kEvalForceLda, kLayD>(c, E, bs, be);
    const long long ni = c->item_off[be] - c->item_off[bs];
    if (ni > 0) {
      FArgs A{};
      if ((rc = density_order(c, bs, be, &A.order))) return rc;
      A.items = c->d_items + c->item_off[bs];
      A.P = E.plane[0]; A.Lp = E.plane[1];
      for (int q = 0; q < 6; q++) A.E[q] = (q < npl - 2) ? E.plane[q + 2] : nullptr;
      A.pad_off = c->d_dpad_off; A.pad_base = c->dpad_off[bs];
      A.D = D_values; A.Q = Q_values; A.F = F; A.max_nnz_pad = c->max_nnz;
      A.ptab_in_smem = c->f_ptab_in_smem ? 1 : 0;
      A.sigma = sigma; A.inv_volume = 1.0 / volume;
      TimedLaunch t(c, kKindForce);
      const int mact = std::max(c->max_act, 1);
      if (sigma) {
        if (g) k_forces<true, true><<<(unsigned)ni, kDThreads, fsm, c->stream>>>(c->S, c->L, A, mact);
        else k_forces<false, true><<<(unsigned)ni, kDThreads, fsm, c->stream>>>(c->S, c->L, A, mact);
      } else {
        if (g) k_forces<true, false><<<(unsigned)ni, kDThreads, fsm, c->stream>>>(c->S, c->L, A, mact);
        else k_forces<false, false><<<(unsigned)ni, kDThreads, fsm, c->stream>>>(c->S, c->L, A, mact);
      }
    }
    if ((rc = check_async(c))) return rc;
    bs = be;
  }
  return AIMS_OK;
}

static int impl_partition_weights(aims_gpu_ctx *c, int64_t n, const double *xyz, const int32_t *owner, double r_part,
                               double *w_part) {
  if (!c || n < 0 || (n && (!xyz || !owner || !w_part)) || !(r_part > 0)) return fail(c, AIMS_ERR_INVALID_ARG, "NULL array, n < 0 or r_part <= 0");
  CU_TRY(c, cudaSetDevice(c->device));
  if (!n) return AIMS_OK;
  // cell list of the atoms, cell edge r_part (a hair more, so that rounding of a cell index never hides a neighbour):
  // every atom within r_part of a point lies in the 27 cells around the point's cell -> O(N) overall.
  // The atoms of a context never change, so the list is kept for the last r_part seen (a grid is usually weighted in several
  // calls with one radius); d_part = [flag word, 63 pad | cell_start | cell_atom].
  if (!(c->part_r == r_part)) {
    const int na = c->S.n_atoms;
    const std::vector<double> &R = c->h_atom_xyz;
    double lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    for (int a = 0; a < na; a++)
      for (int d = 0; d < 3; d++) {
        if (a == 0 || R[3 * a + d] < lo[d]) lo[d] = R[3 * a + d];
        if (a == 0 || R[3 * a + d] > hi[d]) hi[d] = R[3 * a + d];
      }
    const double edge = r_part * (1.0 + 1e-9);
    int dim[3];
    for (int d = 0; d < 3; d++) {
      const double cells = std::floor((hi[d] - lo[d]) / edge) + 1.0;
      if (!(cells < 2048.0)) return fail(c, AIMS_ERR_UNSUPPORTED, "atoms span more than 2048 cells of edge r_part along one axis");
      dim[d] = (int)cells;
    }
    const long long ncell = (long long)dim[0] * dim[1] * dim[2];
    if (ncell > (1ll << 26)) return fail(c, AIMS_ERR_UNSUPPORTED, "cell list of the atoms too large (more than 2^26 cells of edge r_part)");
    std::vector<int> start((size_t)ncell + 1, 0), order((size_t)std::max(na, 1)), cell_of((size_t)std::max(na, 1));
    for (int a = 0; a < na; a++) {
      int ic[3];
      for (int d = 0; d < 3; d++) ic[d] = std::min(dim[d] - 1, std::max(0, (int)std::floor((R[3 * a + d] - lo[d]) / edge)));
      cell_of[a] = (ic[2] * dim[1] + ic[1]) * dim[0] + ic[0];
      start[(size_t)cell_of[a] + 1]++;
    }
    for (long long q = 0; q < ncell; q++) start[(size_t)q + 1] += start[(size_t)q];
    {
      std::vector<int> fill(start.begin(), start.end() - 1);
      for (int a = 0; a < na; a++) order[(size_t)fill[(size_t)cell_of[a]]++] = a;      // ascending atom index inside a cell
    }
    // device copies live in a context-owned buffer that only grows
    const size_t need = 64 + start.size() + order.size();
    c->part_r = -1.0;                                     // nothing cached while the buffer is being replaced
    if (need > c->part_cap) {
      CU_TRY(c, cudaStreamSynchronize(c->stream));
      if (c->d_part) { c->owned.erase(std::remove(c->owned.begin(), c->owned.end(), (void *)c->d_part), c->owned.end()); cudaFree(c->d_part); c->d_part = nullptr; }
      c->part_cap = 0;
      int rc = dev_alloc(c, &c->d_part, need);
      if (rc) return rc;
      c->part_cap = need;
    }
    CU_TRY(c, cudaMemcpyAsync(c->d_part + 64, start.data(), start.size() * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CU_TRY(c, cudaMemcpyAsync(c->d_part + 64 + start.size(), order.data(), order.size() * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));          // start / order are host temporaries
    c->part_cells = PartCells{lo[0], lo[1], lo[2], 1.0 / edge, dim[0], dim[1], dim[2], c->d_part + 64, c->d_part + 64 + start.size()};
    c->part_r = r_part;
  }
  // the kernel raises the flag word for a point with more than kPartMaxCand atoms within r_part (and writes 0 for it): read
  // back here, so that the caller is told by THIS call and not by a later aims_gpu_synchronize
  CU_TRY(c, cudaMemsetAsync(c->d_part, 0, sizeof(int), c->stream));
  {
    TimedLaunch t(c, kKindOther);
    k_partition_weights<<<(unsigned)((n + kPartWarps - 1) / kPartWarps), kPartWarps * 32, 0, c->stream>>>(
        c->part_cells, c->S.atom_xyz, (long long)n, xyz, owner, r_part, w_part, c->d_part);
  }
  int rc = check_async(c);
  if (rc) return rc;
  int flag = 0;
  CU_TRY(c, cudaMemcpyAsync(&flag, c->d_part, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  CU_TRY(c, cudaStreamSynchronize(c->stream));
  if (flag) return fail(c, AIMS_ERR_UNSUPPORTED, "a point has more than 256 atoms within r_part (its weight was set to 0)");
  return AIMS_OK;
}

static int impl_bloch_fold(aims_gpu_ctx *c, const double *H_values, const int32_t *atom_home, const double *atom_T,
                        int32_t n_home, const double *kpt, double *out_re, double *out_im, int accumulate) {
  if (!c || !H_values || !atom_home || !atom_T || !kpt || !out_re || !out_im) return fail(c, AIMS_ERR_INVALID_ARG, "NULL argument");
  const int na = c->S.n_atoms;
  if (n_home <= 0 || n_home > na) return fail(c, AIMS_ERR_INVALID_ARG, "n_home outside [1, n_atoms]");
  for (int a = 0; a < na; a++) {
    const int h = atom_home[a];
    if (h < 0 || h >= n_home || c->h_atom_fn_ptr[h + 1] - c->h_atom_fn_ptr[h] != c->h_atom_fn_ptr[a + 1] - c->h_atom_fn_ptr[a])
      return fail(c, AIMS_ERR_INVALID_ARG, "atom_home must map every atom to a cell atom (< n_home) with the same functions");
  }
  CU_TRY(c, cudaSetDevice(c->device));
  const int nhb = c->h_atom_fn_ptr[n_home];
  // the contribution lists depend on atom_home alone: built once and kept (rebuilt when the caller passes another mapping)
  if (c->bloch_n_home != n_home || c->bloch_home.size() != (size_t)na || !std::equal(c->bloch_home.begin(), c->bloch_home.end(), atom_home)) {
    std::vector<int> cnt((size_t)n_home * n_home + 1, 0);
    for (int A = 0; A < na; A++)
      for (long long q = c->h_row_ptr[A]; q < c->h_row_ptr[A + 1]; q++) {
        const int B = c->h_col_atom[(size_t)q];
        cnt[(size_t)atom_home[A] * n_home + atom_home[B] + 1]++;
        if (A != B) cnt[(size_t)atom_home[B] * n_home + atom_home[A] + 1]++;
      }
    for (size_t t = 0; t + 1 < cnt.size(); t++) cnt[t + 1] += cnt[t];
    std::vector<int> pos(cnt.begin(), cnt.end() - 1);
    std::vector<BlochContrib> contrib((size_t)cnt.back());
    for (int A = 0; A < na; A++)                                   // ascending block index inside every tile: a fixed order
      for (long long q = c->h_row_ptr[A]; q < c->h_row_ptr[A + 1]; q++) {
        const int B = c->h_col_atom[(size_t)q];
        BlochContrib bc{c->h_blk_off[(size_t)q], c->h_blk_ld[(size_t)q], A, B, 0};
        contrib[(size_t)pos[(size_t)atom_home[A] * n_home + atom_home[B]]++] = bc;
        if (A != B) { bc.transposed = 1; contrib[(size_t)pos[(size_t)atom_home[B] * n_home + atom_home[A]]++] = bc; }
      }
    CU_TRY(c, cudaStreamSynchronize(c->stream));                   // nothing in flight may still read the old lists
    for (void *p : {(void *)c->d_bloch_contrib, (void *)c->d_bloch_tile_ptr, (void *)c->d_bloch_T})
      if (p) { c->owned.erase(std::remove(c->owned.begin(), c->owned.end(), p), c->owned.end()); cudaFree(p); }
    c->d_bloch_contrib = nullptr; c->d_bloch_tile_ptr = nullptr; c->d_bloch_T = nullptr; c->bloch_n_home = 0;
    int rc;
    if ((rc = dev_upload<BlochContrib>(c, &c->d_bloch_contrib, contrib.data(), contrib.size()))) return rc;
    if ((rc = dev_upload<int>(c, &c->d_bloch_tile_ptr, cnt.data(), cnt.size()))) return rc;
    if ((rc = dev_alloc(c, &c->d_bloch_T, (size_t)3 * na))) return rc;
    CU_TRY(c, cudaStreamSynchronize(c->stream));                   // contrib / cnt are host temporaries
    c->bloch_home.assign(atom_home, atom_home + na);
    c->bloch_n_home = n_home;
  }
  // atom_T is a HOST array the caller may free after the call: staged through a context-owned copy, then the stream
  // is synchronised (as the header states)
  c->bloch_T_host.assign(atom_T, atom_T + 3 * (size_t)na);
  CU_TRY(c, cudaMemcpyAsync(c->d_bloch_T, c->bloch_T_host.data(), 3 * (size_t)na * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  {
    TimedLaunch t(c, kKindOther);
    k_bloch_fold<<<(unsigned)(n_home * n_home), 128, 0, c->stream>>>(c->d_bloch_contrib, c->d_bloch_tile_ptr, c->S.atom_fn_ptr, c->d_bloch_T,
                                                                  kpt[0], kpt[1], kpt[2], H_values, n_home, nhb, out_re, out_im,
                                                                  accumulate ? 1 : 0);
  }
  cudaError_t e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) { c->err = std::string("aims_gpu_bloch_fold: ") + cudaGetErrorString(e); return AIMS_ERR_CUDA; }
  return check_async(c);
}

static int impl_density_hessian(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *D_values, double *hess_n) {
  if (!range_ok(c, b0, b1)) return fail(c, AIMS_ERR_INVALID_ARG, "batch range outside [0, n_batches]");
  if (!D_values || (!hess_n && c->n_points)) return fail(c, AIMS_ERR_INVALID_ARG, "NULL D_values or hess_n");
  CU_TRY(c, cudaSetDevice(c->device));
  const size_t xsm = x_smem_bytes(c->max_nnz, std::max(c->max_act, 1), c->x_ptab_in_smem);
  if (xsm > c->smem_optin - kStaticSmemMargin) return fail(c, AIMS_ERR_UNSUPPORTED, "nnz(B) too large for the Hessian kernel's shared memory");
  int rc = run_cull(c, b0, b1);
  if (rc) return rc;
  const int npl = 10;
  for (int bs = b0; bs < b1;) {
    const int be = chunk_end(c, c->dpad_off, bs, b1, npl);
    if (be < 0) return fail(c, AIMS_ERR_NOMEM, "workspace too small for one batch of Phi planes");
    const long long plane = (c->ws_doubles / npl) & ~63ll;
    EvalArgs E{};
    for (int q = 0; q < npl; q++) E.plane[q] = c->ws + q * plane;
    E.pad_off = c->d_dpad_off; E.pad_base = c->dpad_off[bs];
    E.n_points = c->n_points;
    launch_eval<kEvalHess, kLayD>(c, E, bs, be);
    const long long ni = c->item_off[be] - c->item_off[bs];
    if (ni > 0) {
      XArgs A{};
      if ((rc = density_order(c, bs, be, &A.order))) return rc;
      A.items = c->d_items + c->item_off[bs];
      for (int q = 0; q < npl; q++) A.PL[q] = E.plane[q];
      A.pad_off = c->d_dpad_off; A.pad_base = c->dpad_off[bs];
      A.D = D_values; A.hn = hess_n; A.n_points = c->n_points; A.max_nnz_pad = c->max_nnz;
      A.ptab_in_smem = c->x_ptab_in_smem ? 1 : 0;
      TimedLaunch t(c, kKindForce);
      k_density_hessian<<<(unsigned)ni, kDThreads, xsm, c->stream>>>(c->S, c->L, A, std::max(c->max_act, 1));
    }
    if ((rc = check_async(c))) return rc;
    bs = be;
  }
  return AIMS_OK;
}

static int impl_pulay_forces(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, const double *D_values,
                          const double *Q_values, double *F, int accumulate) {
  return run_forces(c, b0, b1, v, g, 0, D_values, Q_values, F, accumulate);
}

static int impl_pulay_forces_ks(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, int kinetic,
                             const double *D_values, const double *Q_values, double *F, int accumulate) {
  return run_forces(c, b0, b1, v, g, kinetic, D_values, Q_values, F, accumulate);
}

static int impl_set_deterministic(aims_gpu_ctx *c, int enable) {
  if (!c) return AIMS_ERR_INVALID_ARG;
  c->deterministic = enable != 0;
  return AIMS_OK;
}

static int impl_pulay_forces_stress(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, int kinetic,
                                    const double *D_values, const double *Q_values, double volume, double *F, double *sigma,
                                    int accumulate) {
  if (!sigma) return fail(c, AIMS_ERR_INVALID_ARG, "NULL sigma");
  return run_forces(c, b0, b1, v, g, kinetic, D_values, Q_values, F, accumulate, sigma, volume);
}

static int impl_timing_enable(aims_gpu_ctx *c, int enable) {
  if (!c) return AIMS_ERR_INVALID_ARG;
  CU_TRY(c, cudaSetDevice(c->device));
  CU_TRY(c, cudaStreamSynchronize(c->stream));
  for (auto &sp : c->spans) c->pool.push_back(sp);
  c->spans.clear();
  c->timing = enable != 0;
  return AIMS_OK;
}

static int impl_timing_read(aims_gpu_ctx *c, double *ms, int64_t *launches) {
  if (!c || !ms || !launches) return AIMS_ERR_INVALID_ARG;
  CU_TRY(c, cudaSetDevice(c->device));
  CU_TRY(c, cudaStreamSynchronize(c->stream));
  for (int k = 0; k < kNumKinds; k++) { ms[k] = 0.0; launches[k] = 0; }
  cudaError_t bad = cudaSuccess;
  for (auto &sp : c->spans) {
    float t = 0.f;
    const cudaError_t e = cudaEventElapsedTime(&t, sp.e0, sp.e1);
    if (e != cudaSuccess) bad = e;
    else { ms[sp.kind] += t; launches[sp.kind]++; }
    c->pool.push_back(sp);          // every span goes back to the pool exactly once, also on an error
  }
  c->spans.clear();
  if (bad != cudaSuccess) { c->err = std::string("cudaEventElapsedTime: ") + cudaGetErrorString(bad); return AIMS_ERR_CUDA; }
  return AIMS_OK;
}

static int impl_synchronize(aims_gpu_ctx *c) {
  if (!c) return AIMS_ERR_INVALID_ARG;
  CU_TRY(c, cudaSetDevice(c->device));
  int flag = 0;
  CU_TRY(c, cudaMemcpyAsync(&flag, c->L.error_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  CU_TRY(c, cudaStreamSynchronize(c->stream));
  if (flag) {
    // reported once: the flag is cleared, so that a later synchronize reports only what was flagged since
    CU_TRY(c, cudaMemsetAsync(c->L.error_flag, 0, sizeof(int), c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    c->err = "device-side capacity or consistency check failed (flag " + std::to_string(flag) + ")";
    return AIMS_ERR_UNSUPPORTED;
  }
  return AIMS_OK;
}

#ifdef AIMS_PROBE_DMMA
static int impl_dmma_probe(aims_gpu_ctx *c, int variant, int warps_per_sm, double *tflops) {
  if (!c || !tflops || variant < 1 || variant > 11 || warps_per_sm < 1 || warps_per_sm > (variant <= 3 ? 16 : 20))
    return fail(c, AIMS_ERR_INVALID_ARG, "variant 1..11, warps_per_sm 1..16 (variants 4..11: 1..20)");
  CU_TRY(c, cudaSetDevice(c->device));
  if (!c->probe_out) { int rc = dev_alloc(c, &c->probe_out, 16); if (rc) return rc; }   // scratch of the probes, allocated once
  double *out = c->probe_out;
  const int iters = 40000, threads = 32 * warps_per_sm;
  if (variant >= 10) {   // trip counts of k_dmma_probe3 live in global memory: 10,000 stages of 4 steps
    const int cnt[2] = {iters / 4, (iters / 4) * 16};
    CU_TRY(c, cudaMemcpyAsync(out + 8, cnt, sizeof(cnt), cudaMemcpyHostToDevice, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
  }
  cudaEvent_t e0, e1;
  CU_TRY(c, cudaEventCreate(&e0));
  CU_TRY(c, cudaEventCreate(&e1));
  for (int rep = 0; rep < 2; rep++) {          // the first launch warms up
    if (rep == 1) CU_TRY(c, cudaEventRecord(e0, c->stream));
    if (variant == 1) k_dmma_probe<1><<<c->sm_count, threads, 0, c->stream>>>(out, iters, 1.0000001, 1e-9);
    else if (variant == 2) k_dmma_probe<2><<<c->sm_count, threads, 0, c->stream>>>(out, iters, 1.0000001, 1e-9);
    else if (variant == 3) k_dmma_probe<3><<<c->sm_count, threads, 0, c->stream>>>(out, iters, 1.0000001, 1e-9);
    else if (variant == 4) k_dmma_probe2<4, 4, true><<<c->sm_count, threads, 0, c->stream>>>(out, iters, 1e-9);
    else if (variant == 5) k_dmma_probe2<4, 3, true><<<c->sm_count, threads, 0, c->stream>>>(out, iters, 1e-9);
    else if (variant == 6) k_dmma_probe2<3, 3, true><<<c->sm_count, threads, 0, c->stream>>>(out, iters, 1e-9);
    else if (variant == 7) k_dmma_probe2<4, 4, false><<<c->sm_count, threads, 0, c->stream>>>(out, iters, 1e-9);
    else if (variant == 8) k_dmma_probe2<4, 3, false><<<c->sm_count, threads, 0, c->stream>>>(out, iters, 1e-9);
    else if (variant == 9) k_dmma_probe2<2, 2, true><<<c->sm_count, threads, 0, c->stream>>>(out, iters, 1e-9);
    else if (variant == 10) k_dmma_probe3<false><<<c->sm_count, threads, 0, c->stream>>>(out, reinterpret_cast<const int *>(out + 8), 1e-9);
    else k_dmma_probe3<true><<<c->sm_count, threads, 0, c->stream>>>(out, reinterpret_cast<const int *>(out + 8), 1e-9);
    c->launches++;
  }
  CU_TRY(c, cudaEventRecord(e1, c->stream));
  CU_TRY(c, cudaEventSynchronize(e1));
  float ms = 0;
  CU_TRY(c, cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  const int per_step[12] = {0, 16, 16, 16, 16, 12, 9, 16, 12, 4, 12, 12};        // DMMAs per step and warp
  *tflops = 2.0 * 256 * per_step[variant] * (double)iters * c->sm_count * warps_per_sm / (ms * 1e-3) * 1e-12;
  return check_async(c);
}
#else
static int impl_dmma_probe(aims_gpu_ctx *c, int, int, double *) {
  return fail(c, AIMS_ERR_UNSUPPORTED, "aims_gpu_dmma_probe: the operand-pattern probes are compiled into probe builds only "
                                       "(python -m paper_1912_06636_b200.build --define AIMS_PROBE_DMMA=1 --tag dmma)");
}
#endif

static int impl_fp64_peak(aims_gpu_ctx *c, double ms_target, double *tflops) {
  if (!c || !tflops) return AIMS_ERR_INVALID_ARG;
  CU_TRY(c, cudaSetDevice(c->device));
  if (!c->probe_out) { int rc = dev_alloc(c, &c->probe_out, 16); if (rc) return rc; }   // scratch of the probes, allocated once
  double *out = c->probe_out;
  const int iters = 20000;
  const dim3 grid(c->sm_count), block(256);
  cudaEvent_t e0, e1;
  CU_TRY(c, cudaEventCreate(&e0));
  CU_TRY(c, cudaEventCreate(&e1));
  k_fp64_peak<<<grid, block, 0, c->stream>>>(out, iters, 1.0000001, 1e-9);  // warm-up, ~5 ms
  c->launches++;
  const int reps = std::max(1, (int)(ms_target / 5.3));
  CU_TRY(c, cudaEventRecord(e0, c->stream));
  for (int r = 0; r < reps; r++) k_fp64_peak<<<grid, block, 0, c->stream>>>(out, iters, 1.0000001, 1e-9);
  c->launches += reps;
  CU_TRY(c, cudaEventRecord(e1, c->stream));
  CU_TRY(c, cudaEventSynchronize(e1));
  float ms = 0;
  CU_TRY(c, cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *tflops = 2.0 * 256 * 16 * (double)iters * grid.x * (block.x / 32) * reps / (ms * 1e-3) * 1e-12;
  return AIMS_OK;
}

}  // extern "C"

// ---- aims_gpu_partition_weights_noalloc: k_partition_weights for callers that cannot allocate device memory (an MPS client at
// its memory limit, a program whose pool allocator owns the HBM, a loop that must not stall in cudaMalloc).  What
// impl_partition_weights keeps in a cudaMalloc'ed buffer of the context -- flag word, cell_start, cell_atom -- and what it
// borrows from the context -- the device copy of the atom positions -- sits here in ONE array that is part of the library
// image: every device that loads the library carries these 1.5 MB until the process ends.  The sizes the array is cut for
// are the limits in include/aims_gpu.h.
//
// `g_noalloc_scratch` names the array in DEVICE code.  In host code the same name is only the handle the runtime registered for
// it -- not an address a kernel may dereference -- so the host asks the runtime, per device, where the array actually lives
// (noalloc_scratch_on) and passes that pointer to the kernel.
constexpr size_t kNaCellStartBytes = 4 * ((size_t)AIMS_NOALLOC_MAX_CELLS + 64);    // int [cells + 1], rounded up to 256 B
constexpr size_t kNaCellAtomBytes = 4 * (size_t)AIMS_NOALLOC_MAX_ATOMS;            // int [atoms]
constexpr size_t kNaAtomXyzBytes = 24 * (size_t)AIMS_NOALLOC_MAX_ATOMS;            // double [atoms][3]
constexpr size_t kNaOffCellAtom = kNaCellStartBytes, kNaOffAtomXyz = kNaOffCellAtom + kNaCellAtomBytes,
                 kNaOffFlag = kNaOffAtomXyz + kNaAtomXyzBytes, kNaBytes = kNaOffFlag + 256;
static_assert(kNaBytes == AIMS_NOALLOC_SCRATCH_BYTES, "header states the size of the array");
static_assert(kNaOffCellAtom % 256 == 0 && kNaOffAtomXyz % 256 == 0 && kNaOffFlag % 256 == 0, "sub-arrays keep the alignment");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNaBytes];

namespace {

constexpr int kNaMaxDevices = 64;
std::mutex g_noalloc_mu;
unsigned char *g_noalloc_ptr[kNaMaxDevices] = {};   // device address of g_noalloc_scratch, per device ordinal (0 = not asked yet)

// Set-up, once per device and process: `device` must be current.  The first use of a symbol of this module may make the
// runtime load the module, which is why the header asks for the first call to come before any stream capture.
cudaError_t noalloc_scratch_on(int device, unsigned char **out) {
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[device]) {
    void *p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_noalloc_ptr[device] = static_cast<unsigned char *>(p);
  }
  *out = g_noalloc_ptr[device];
  return cudaSuccess;
}

int na_fail(char *err_text, int cap, int code, const char *fmt, ...) {
  if (err_text && cap > 0) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(err_text, (size_t)cap, fmt, ap);
    va_end(ap);
  }
  return code;
}

#define NA_TRY(call)                                                                                            \
  do {                                                                                                          \
    const cudaError_t e_ = (call);                                                                              \
    if (e_ != cudaSuccess) return na_fail(err_text, cap, AIMS_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

int impl_partition_weights_noalloc(int device, cudaStream_t st, int na, const double *R, long long n, const double *xyz,
                                   const int *owner, double r_part, double *w_part, char *err_text, int cap) {
  if (err_text && cap > 0) err_text[0] = 0;
  if (device < 0 || device >= kNaMaxDevices || na < 0 || n < 0 || (na && !R) || (n && (!xyz || !owner || !w_part)) || !(r_part > 0))
    return na_fail(err_text, cap, AIMS_ERR_INVALID_ARG, "NULL array, negative size, r_part <= 0 or device outside [0, %d)", kNaMaxDevices);
  if (na > AIMS_NOALLOC_MAX_ATOMS)
    return na_fail(err_text, cap, AIMS_ERR_UNSUPPORTED, "n_atoms = %d is more than AIMS_NOALLOC_MAX_ATOMS = %d, the size the built-in scratch "
                   "array is cut for; use aims_gpu_partition_weights (it allocates)", na, AIMS_NOALLOC_MAX_ATOMS);
  if (!n) return AIMS_OK;
  // cell list of the atoms on the host, as in impl_partition_weights: edge a hair above r_part, atoms ascending inside a cell
  double lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
  for (int a = 0; a < na; a++)
    for (int d = 0; d < 3; d++) {
      if (!std::isfinite(R[3 * a + d])) return na_fail(err_text, cap, AIMS_ERR_INVALID_ARG, "atom_xyz[%d][%d] is not finite", a, d);
      if (a == 0 || R[3 * a + d] < lo[d]) lo[d] = R[3 * a + d];
      if (a == 0 || R[3 * a + d] > hi[d]) hi[d] = R[3 * a + d];
    }
  const double edge = r_part * (1.0 + 1e-9);
  int dim[3];
  double cells_total = 1.0;
  for (int d = 0; d < 3; d++) {
    const double cells = std::floor((hi[d] - lo[d]) / edge) + 1.0;
    cells_total *= cells;
    dim[d] = cells <= (double)AIMS_NOALLOC_MAX_CELLS ? (int)cells : 0;
  }
  if (!(cells_total <= (double)AIMS_NOALLOC_MAX_CELLS))
    return na_fail(err_text, cap, AIMS_ERR_UNSUPPORTED, "the atoms span %.0f cells of edge r_part = %g, more than AIMS_NOALLOC_MAX_CELLS = %d, the "
                   "size the built-in scratch array is cut for; use aims_gpu_partition_weights (it allocates)", cells_total, r_part,
                   AIMS_NOALLOC_MAX_CELLS);
  const int ncell = dim[0] * dim[1] * dim[2];
  std::vector<int> start((size_t)ncell + 1, 0), order((size_t)std::max(na, 1)), cell_of((size_t)std::max(na, 1));
  for (int a = 0; a < na; a++) {
    int ic[3];
    for (int d = 0; d < 3; d++) ic[d] = std::min(dim[d] - 1, std::max(0, (int)std::floor((R[3 * a + d] - lo[d]) / edge)));
    cell_of[a] = (ic[2] * dim[1] + ic[1]) * dim[0] + ic[0];
    start[(size_t)cell_of[a] + 1]++;
  }
  for (int q = 0; q < ncell; q++) start[(size_t)q + 1] += start[(size_t)q];
  {
    std::vector<int> fill(start.begin(), start.end() - 1);
    for (int a = 0; a < na; a++) order[(size_t)fill[(size_t)cell_of[a]]++] = a;
  }

  NA_TRY(cudaSetDevice(device));
  unsigned char *base = nullptr;
  NA_TRY(noalloc_scratch_on(device, &base));
  int *d_start = reinterpret_cast<int *>(base), *d_order = reinterpret_cast<int *>(base + kNaOffCellAtom),
      *d_flag = reinterpret_cast<int *>(base + kNaOffFlag);
  double *d_R = reinterpret_cast<double *>(base + kNaOffAtomXyz);
  // the array still holds the previous call's cell list and flag: everything the kernel reads is overwritten here, and the
  // flag -- which the kernel only ever raises -- is cleared
  NA_TRY(cudaMemcpyAsync(d_start, start.data(), start.size() * sizeof(int), cudaMemcpyHostToDevice, st));
  if (na) {
    NA_TRY(cudaMemcpyAsync(d_order, order.data(), (size_t)na * sizeof(int), cudaMemcpyHostToDevice, st));
    NA_TRY(cudaMemcpyAsync(d_R, R, (size_t)na * 3 * sizeof(double), cudaMemcpyHostToDevice, st));
  }
  NA_TRY(cudaMemsetAsync(d_flag, 0, sizeof(int), st));
  const PartCells PC{lo[0], lo[1], lo[2], 1.0 / edge, dim[0], dim[1], dim[2], d_start, d_order};
  k_partition_weights<<<(unsigned)((n + kPartWarps - 1) / kPartWarps), kPartWarps * 32, 0, st>>>(PC, d_R, n, xyz, owner, r_part, w_part, d_flag);
  NA_TRY(cudaGetLastError());
  int flag = 0;
  NA_TRY(cudaMemcpyAsync(&flag, d_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
  NA_TRY(cudaStreamSynchronize(st));                     // start / order / R are the caller's or host temporaries; flag is read here
  if (flag)
    return na_fail(err_text, cap, AIMS_ERR_UNSUPPORTED, "a point has more than %d atoms within r_part = %g (its weight was set to 0)", kPartMaxCand, r_part);
  return AIMS_OK;
}

}  // namespace

// ---- the exported entry points: every body runs under `guarded` (no exception leaves the library)
extern "C" {

int aims_gpu_partition_weights_noalloc(int device, void *cuda_stream, int32_t n_atoms, const double *atom_xyz, int64_t n, const double *xyz,
                                       const int32_t *owner, double r_part, double *w_part, char *err_text, int32_t err_capacity) {
  const int rc = guarded(nullptr, [&] {
    return impl_partition_weights_noalloc(device, static_cast<cudaStream_t>(cuda_stream), n_atoms, atom_xyz, (long long)n, xyz, owner, r_part,
                                          w_part, err_text, err_capacity);
  });
  if (rc == AIMS_ERR_NOMEM && err_text && err_capacity > 0 && !err_text[0]) snprintf(err_text, (size_t)err_capacity, "out of host memory");
  return rc;
}

int aims_gpu_create(aims_gpu_ctx **out, const aims_basis_desc *B, const aims_grid_desc *G, const aims_bsr_desc *P, int device, void *cuda_stream, int64_t workspace_bytes) {
  // on failure *out is either NULL or a context that only aims_gpu_last_error and aims_gpu_destroy accept
  const int rc = guarded(nullptr, [&] { return impl_create(out, B, G, P, device, cuda_stream, workspace_bytes); });
  if (rc == AIMS_ERR_NOMEM && out && *out) guarded(nullptr, [&] { if ((*out)->err.empty()) (*out)->err = "out of memory"; return 0; });
  return rc;
}

int aims_gpu_stats(aims_gpu_ctx *c, int64_t *sum_nnz, int32_t *max_nnz, int32_t *max_active_atoms, double *flops_h_lda, double *flops_h_gga, double *flops_density) {
  return guarded(c, [&] { return impl_stats(c, sum_nnz, max_nnz, max_active_atoms, flops_h_lda, flops_h_gga, flops_density); });
}

int aims_gpu_batch_nnz(aims_gpu_ctx *c, int32_t *nnz) {
  return guarded(c, [&] { return impl_batch_nnz(c, nnz); });
}

int aims_gpu_basis_sizes(aims_gpu_ctx *c, int32_t b0, int32_t b1, int64_t *n_index, int64_t *n_phi) {
  return guarded(c, [&] { return impl_basis_sizes(c, b0, b1, n_index, n_phi); });
}

int aims_gpu_eval_basis(aims_gpu_ctx *c, int32_t b0, int32_t b1, int64_t *fn_ptr, int32_t *fn_index, int64_t *phi_ptr, double *phi, double *dphi) {
  return guarded(c, [&] { return impl_eval_basis(c, b0, b1, fn_ptr, fn_index, phi_ptr, phi, dphi); });
}

int aims_gpu_add_tau_matrix(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *xi, double *H_values) {
  return guarded(c, [&] { return impl_add_tau_matrix(c, b0, b1, xi, H_values); });
}

int aims_gpu_integrate_hamiltonian(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, double *H_values, int accumulate) {
  return guarded(c, [&] { return impl_integrate_hamiltonian(c, b0, b1, v, g, H_values, accumulate); });
}

int aims_gpu_integrate_hamiltonian_ks(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, int kinetic, double *H_values, int accumulate) {
  return guarded(c, [&] { return impl_integrate_hamiltonian_ks(c, b0, b1, v, g, kinetic, H_values, accumulate); });
}

int aims_gpu_update_density(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *D_values, double *n, double *grad_n) {
  return guarded(c, [&] { return impl_update_density(c, b0, b1, D_values, n, grad_n); });
}

int aims_gpu_partition_weights(aims_gpu_ctx *c, int64_t n, const double *xyz, const int32_t *owner, double r_part, double *w_part) {
  return guarded(c, [&] { return impl_partition_weights(c, n, xyz, owner, r_part, w_part); });
}

int aims_gpu_bloch_fold(aims_gpu_ctx *c, const double *H_values, const int32_t *atom_home, const double *atom_T, int32_t n_home, const double *kpt, double *out_re, double *out_im, int accumulate) {
  return guarded(c, [&] { return impl_bloch_fold(c, H_values, atom_home, atom_T, n_home, kpt, out_re, out_im, accumulate); });
}

int aims_gpu_density_hessian(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *D_values, double *hess_n) {
  return guarded(c, [&] { return impl_density_hessian(c, b0, b1, D_values, hess_n); });
}

int aims_gpu_pulay_forces(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, const double *D_values, const double *Q_values, double *F, int accumulate) {
  return guarded(c, [&] { return impl_pulay_forces(c, b0, b1, v, g, D_values, Q_values, F, accumulate); });
}

int aims_gpu_pulay_forces_ks(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, int kinetic, const double *D_values, const double *Q_values, double *F, int accumulate) {
  return guarded(c, [&] { return impl_pulay_forces_ks(c, b0, b1, v, g, kinetic, D_values, Q_values, F, accumulate); });
}

int aims_gpu_pulay_forces_stress(aims_gpu_ctx *c, int32_t b0, int32_t b1, const double *v, const double *g, int kinetic, const double *D_values, const double *Q_values, double volume, double *F, double *sigma, int accumulate) {
  return guarded(c, [&] { return impl_pulay_forces_stress(c, b0, b1, v, g, kinetic, D_values, Q_values, volume, F, sigma, accumulate); });
}

int aims_gpu_set_deterministic(aims_gpu_ctx *c, int enable) {
  return guarded(c, [&] { return impl_set_deterministic(c, enable); });
}

int aims_gpu_timing_enable(aims_gpu_ctx *c, int enable) {
  return guarded(c, [&] { return impl_timing_enable(c, enable); });
}

int aims_gpu_timing_read(aims_gpu_ctx *c, double *ms, int64_t *launches) {
  return guarded(c, [&] { return impl_timing_read(c, ms, launches); });
}

int aims_gpu_synchronize(aims_gpu_ctx *c) {
  return guarded(c, [&] { return impl_synchronize(c); });
}

#ifndef AIMS_BUILD_FLAGS
#define AIMS_BUILD_FLAGS ""        // build.py sets it to the -D list of a probe build
#endif
const char *aims_gpu_build_flags(void) { return AIMS_BUILD_FLAGS; }

int aims_gpu_dmma_probe(aims_gpu_ctx *c, int variant, int warps_per_sm, double *tflops) {
  return guarded(c, [&] { return impl_dmma_probe(c, variant, warps_per_sm, tflops); });
}

int aims_gpu_fp64_peak(aims_gpu_ctx *c, double ms_target, double *tflops) {
  return guarded(c, [&] { return impl_fp64_peak(c, ms_target, tflops); });
}

}  // extern "C"
