// batching.cu -- aims_gpu_batch_points: the grid-adapted cut-plane batching of PAPER.md L210-218 ("Algorithm 3 of [37]":
// the point cloud is bisected by cut planes until a targeted number of points per subset is reached) on the GPU
// (SURVEY.md 8(f) row f4).  The paper only cites the algorithm; reading P12 fixes a deterministic one:
//   a set of n points is a batch if n <= max_pts; else with nb = ceil(n / max_pts) the n_left = round(floor(nb/2) n / nb)
//   points smallest in (coordinate along the axis of largest extent, original index) go left, the rest right; children in
//   depth-first order; a batch keeps the order of its parent's sort.
// Sizes depend on n only, so the host knows the whole tree (batch_ptr) up front; the device finds the ORDER.
//
// k-d-tree construction by presorting, level by level (every segment of a level in the same launches):
//   once     three index arrays perm_c, each sorted by (coordinate c, original index)  [LSD radix sort, stable]
//   a level  every segment occupies the same range [start, start + count) in all three arrays, sorted by c in perm_c, so
//            * its extent along c is coord(perm_c[last]) - coord(perm_c[first])  -> cut axis, no reduction needed,
//            * the first n_left entries of its range in perm_axis are the left child               -> side[point],
//            * a STABLE partition of its range in each perm_c by side[] keeps both children sorted by c
//              (position = start + number of left points before me, from one exclusive prefix sum over the whole array).
// A leaf's final order is its range in perm_(axis of its parent's cut).
#include "../../include/aims_gpu.h"

#include <algorithm>
#include <cstdint>
#include <new>
#include <vector>

#include <cub/device/device_radix_sort.cuh>
#include <cuda_runtime.h>

namespace {

struct Seg { long long start, count, n_left; int parent_axis_slot; int split; };   // one segment of a level

// ---------------------------------------------------------------------------------------------- prefix sum (hand-written)
constexpr int kScanBlock = 1024;       // elements per block: 256 threads x 4

__global__ void __launch_bounds__(256) k_scan_blocks(const unsigned char *flag, int *out, int *block_sum, long long n) {
  __shared__ int s_warp[8];
  const long long base = (long long)blockIdx.x * kScanBlock + threadIdx.x * 4;
  int v[4], t = 0;
#pragma unroll
  for (int k = 0; k < 4; k++) { v[k] = (base + k < n) ? flag[base + k] : 0; t += v[k]; }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int incl = t;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += u; }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  int woff = 0;
  for (int w2 = 0; w2 < warp; w2++) woff += s_warp[w2];
  int run = woff + incl - t;                                   // exclusive prefix of this thread inside the block
#pragma unroll
  for (int k = 0; k < 4; k++) { if (base + k < n) out[base + k] = run; run += v[k]; }
  if (threadIdx.x == 255) block_sum[blockIdx.x] = woff + incl;
}

// exclusive scan of up to 1024 x 1024 block sums by ONE block (n_blocks <= 2^20), in place
__global__ void __launch_bounds__(1024) k_scan_sums(int *block_sum, int n_blocks) {
  __shared__ int s[1024];
  __shared__ int carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < n_blocks; base += 1024) {
    const int i = base + threadIdx.x;
    const int v = i < n_blocks ? block_sum[i] : 0;
    s[threadIdx.x] = v;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
      const int u = threadIdx.x >= o ? s[threadIdx.x - o] : 0;
      __syncthreads();
      s[threadIdx.x] += u;
      __syncthreads();
    }
    if (i < n_blocks) block_sum[i] = carry + s[threadIdx.x] - v;
    __syncthreads();
    if (threadIdx.x == 1023) carry += s[1023];
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------------------- the levels
__device__ __forceinline__ int find_seg(const Seg *segs, int n_segs, long long pos) {
  int lo = 0, hi = n_segs - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (segs[mid].start <= pos) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// the same for a whole block of consecutive positions: one binary search for the block's first position, then every thread walks
// forward from there (a segment that still splits has more than max_pts points, so a block of 256 positions spans a few segments;
// per-thread binary searches over up to 40,000 segments were most of the time of a level on a 7.9 M point grid)
__device__ __forceinline__ int find_seg_block(const Seg *segs, int n_segs, long long pos, long long n) {
  __shared__ int s_first;
  if (threadIdx.x == 0) s_first = find_seg(segs, n_segs, min((long long)blockIdx.x * blockDim.x, n - 1));
  __syncthreads();
  int s = s_first;
  while (s + 1 < n_segs && segs[s + 1].start <= pos) s++;
  return s;
}

__global__ void k_keys(const double *xyz, long long n, int c, double *key, int *idx) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  key[i] = xyz[3 * i + c] + 0.0;          // -0.0 -> +0.0: the two compare equal in the definition
  idx[i] = (int)i;
}

// cut axis of every splitting segment: largest extent, ties to the lower axis (x, then y, then z)
__global__ void k_axis(const Seg *segs, int n_segs, const double *xyz, const int *p0, const int *p1, const int *p2, int *axis) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n_segs) return;
  const Seg g = segs[s];
  if (!g.split) { axis[s] = -1; return; }
  const long long a = g.start, b = g.start + g.count - 1;
  const double e0 = xyz[3ll * p0[b]] - xyz[3ll * p0[a]], e1 = xyz[3ll * p1[b] + 1] - xyz[3ll * p1[a] + 1],
               e2 = xyz[3ll * p2[b] + 2] - xyz[3ll * p2[a] + 2];
  int ax = 0;
  double e = e0;
  if (e1 > e) { ax = 1; e = e1; }
  if (e2 > e) ax = 2;
  axis[s] = ax;
}

// side of every point of a splitting segment (0 = left child), read off its rank in perm_axis
__global__ void k_mark(const Seg *segs, int n_segs, const int *axis, const int *p0, const int *p1, const int *p2, long long n,
                       unsigned char *side) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int s = find_seg_block(segs, n_segs, min(i, n - 1), n);
  if (i >= n) return;
  const Seg g = segs[s];
  if (!g.split) return;
  const int ax = axis[s];
  const int pt = ax == 0 ? p0[i] : ax == 1 ? p1[i] : p2[i];
  side[pt] = (i - g.start) < g.n_left ? 0 : 1;
}

__global__ void k_flags(const int *perm, const unsigned char *side, long long n, unsigned char *flag) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) flag[i] = side[perm[i]] == 0 ? 1 : 0;
}

// stable partition of every splitting segment's range of `perm` by side[]; other ranges are copied
__global__ void k_partition(const Seg *segs, int n_segs, const int *perm, const unsigned char *side, const int *scan,
                            const int *block_sum, long long n, int *perm_out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int s = find_seg_block(segs, n_segs, min(i, n - 1), n);
  if (i >= n) return;
  const Seg g = segs[s];
  const int pt = perm[i];
  if (!g.split) { perm_out[i] = pt; return; }
  auto lefts_before = [&](long long pos) { return (long long)scan[pos] + block_sum[pos / kScanBlock]; };
  const long long lb = lefts_before(i) - lefts_before(g.start);        // left points of the segment before position i
  const long long dst = side[pt] == 0 ? g.start + lb : g.start + g.n_left + ((i - g.start) - lb);
  perm_out[dst] = pt;
}

// a finished level: leaves take their final order from perm_(parent's axis); tag[pos] = axis array to read at the end
__global__ void k_tag_children(const Seg *segs, int n_segs, const int *axis, long long n, signed char *tag) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int s = find_seg_block(segs, n_segs, min(i, n - 1), n);
  if (i >= n) return;
  if (segs[s].split) tag[i] = (signed char)axis[s];
}

__global__ void k_emit(const signed char *tag, const int *p0, const int *p1, const int *p2, long long n, long long *order) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int t = tag[i];
  order[i] = t == 0 ? p0[i] : t == 1 ? p1[i] : t == 2 ? p2[i] : i;
}

long long n_left_of(long long n, int max_pts) {
  const long long nb = (n + max_pts - 1) / max_pts, h = nb / 2;
  return (2 * h * n + nb) / (2 * nb);                          // round(h n / nb), halves up
}

void leaf_sizes(long long lo, long long n, int max_pts, std::vector<long long> &ptr) {
  if (n <= max_pts) { ptr.push_back(lo); return; }
  const long long nl = n_left_of(n, max_pts);
  leaf_sizes(lo, nl, max_pts, ptr);
  leaf_sizes(lo + nl, n - nl, max_pts, ptr);
}

struct DevBuf {
  std::vector<void *> owned;
  ~DevBuf() { for (void *p : owned) cudaFree(p); }
  template <class T>
  cudaError_t get(T **p, size_t n) {
    void *q = nullptr;
    cudaError_t e = cudaMalloc(&q, std::max<size_t>(n, 1) * sizeof(T));
    if (e == cudaSuccess) owned.push_back(q);
    *p = static_cast<T *>(q);
    return e;
  }
};

#define BT(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return e_ == cudaErrorMemoryAllocation ? AIMS_ERR_NOMEM : AIMS_ERR_CUDA; } while (0)

int batch_points_impl(int device, cudaStream_t st, long long n, const double *xyz, int max_pts, long long *order,
                      long long *batch_ptr, long long cap, int *n_batches) {
  if (n < 0 || max_pts <= 0 || !batch_ptr || !n_batches || cap < 1 || (n && (!xyz || !order)) || n >= (1ll << 31))
    return AIMS_ERR_INVALID_ARG;
  // the tree shape depends on n only (host)
  std::vector<long long> ptr;
  if (n > 0) leaf_sizes(0, n, max_pts, ptr);
  ptr.push_back(n);
  if ((long long)ptr.size() > cap) return AIMS_ERR_INVALID_ARG;
  *n_batches = (int)ptr.size() - 1;
  std::copy(ptr.begin(), ptr.end(), batch_ptr);
  if (n == 0) return AIMS_OK;
  BT(cudaSetDevice(device));
  const unsigned gb = (unsigned)((n + 255) / 256);
  DevBuf D;
  signed char *tag;
  BT(D.get(&tag, (size_t)n));
  BT(cudaMemsetAsync(tag, 0xFF, (size_t)n, st));                 // -1: identity (a root that is itself a batch)
  int *perm[3] = {nullptr, nullptr, nullptr}, *perm_alt;
  for (int c = 0; c < 3; c++) BT(D.get(&perm[c], (size_t)n));
  BT(D.get(&perm_alt, (size_t)n));
  if (n > max_pts) {
    // ---- three presorted index arrays
    double *key, *key_out;
    int *idx;
    BT(D.get(&key, (size_t)n)); BT(D.get(&key_out, (size_t)n)); BT(D.get(&idx, (size_t)n));
    size_t tmp_bytes = 0;
    BT(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, key, key_out, idx, perm[0], (int)n, 0, 64, st));
    unsigned char *tmp;
    BT(D.get(&tmp, tmp_bytes));
    for (int c = 0; c < 3; c++) {
      k_keys<<<gb, 256, 0, st>>>(xyz, n, c, key, idx);
      BT(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, key, key_out, idx, perm[c], (int)n, 0, 64, st));   // stable
    }
    // ---- levels
    unsigned char *side, *flag;
    int *scan, *bsum, *axis;
    Seg *d_segs;
    const int n_blocks = (int)((n + kScanBlock - 1) / kScanBlock);
    BT(D.get(&side, (size_t)n)); BT(D.get(&flag, (size_t)n)); BT(D.get(&scan, (size_t)n)); BT(D.get(&bsum, (size_t)n_blocks + 1));
    BT(D.get(&axis, (size_t)*n_batches + 1)); BT(D.get(&d_segs, (size_t)*n_batches + 1));
    std::vector<Seg> level{Seg{0, n, 0, -1, 0}};
    while (true) {
      bool any = false;
      for (Seg &g : level) { g.split = g.count > max_pts; g.n_left = g.split ? n_left_of(g.count, max_pts) : 0; any |= g.split != 0; }
      if (!any) break;
      const int ns = (int)level.size();
      BT(cudaMemcpyAsync(d_segs, level.data(), ns * sizeof(Seg), cudaMemcpyHostToDevice, st));
      k_axis<<<(ns + 127) / 128, 128, 0, st>>>(d_segs, ns, xyz, perm[0], perm[1], perm[2], axis);
      k_mark<<<gb, 256, 0, st>>>(d_segs, ns, axis, perm[0], perm[1], perm[2], n, side);
      k_tag_children<<<gb, 256, 0, st>>>(d_segs, ns, axis, n, tag);
      for (int c = 0; c < 3; c++) {
        k_flags<<<gb, 256, 0, st>>>(perm[c], side, n, flag);
        k_scan_blocks<<<n_blocks, 256, 0, st>>>(flag, scan, bsum, n);
        k_scan_sums<<<1, 1024, 0, st>>>(bsum, n_blocks);
        k_partition<<<gb, 256, 0, st>>>(d_segs, ns, perm[c], side, scan, bsum, n, perm_alt);
        std::swap(perm[c], perm_alt);
      }
      BT(cudaStreamSynchronize(st));                             // `level` is re-built below while d_segs may still be read
      std::vector<Seg> next;
      next.reserve(level.size() * 2);
      for (const Seg &g : level) {
        if (!g.split) { next.push_back(g); continue; }
        next.push_back(Seg{g.start, g.n_left, 0, -1, 0});
        next.push_back(Seg{g.start + g.n_left, g.count - g.n_left, 0, -1, 0});
      }
      level.swap(next);
    }
  }
  k_emit<<<gb, 256, 0, st>>>(tag, perm[0], perm[1], perm[2], n, order);
  BT(cudaGetLastError());
  BT(cudaStreamSynchronize(st));                                 // the scratch buffers are freed on return
  return AIMS_OK;
}

}  // namespace

extern "C" int aims_gpu_batch_points(int device, void *cuda_stream, int64_t n_points, const double *xyz, int32_t max_batch_points,
                                     int64_t *order, int64_t *batch_ptr, int64_t batch_ptr_capacity, int32_t *n_batches) {
  try {
    static_assert(sizeof(long long) == sizeof(int64_t), "int64_t is long long here");
    return batch_points_impl(device, static_cast<cudaStream_t>(cuda_stream), n_points, xyz, max_batch_points,
                             reinterpret_cast<long long *>(order), reinterpret_cast<long long *>(batch_ptr), batch_ptr_capacity,
                             n_batches);
  } catch (const std::bad_alloc &) {
    return AIMS_ERR_NOMEM;
  } catch (...) {
    return AIMS_ERR_INVALID_ARG;
  }
}
