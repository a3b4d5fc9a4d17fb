// gale_init.cuh — device side of the initialization ("Initialization": the interval
// array I_T, the external lists T_ex per segment; here also the tile-local re-encoding the batch kernels
// stage). The paper builds these on the CPU; here the simplices never leave the GPU:
// every pass over T or over the vertices is a kernel, the host only handles per-tile / per-cluster
// scalars (prefix sums over a few hundred thousand tiles).
#pragma once
#include <cuda_runtime.h>
#include <limits.h>
#include <stdint.h>

#include "gale_kernels.cuh"

namespace gale {
namespace init {

// C1-C3 of the input contract (rows strictly ascending, rows strictly ascending lexicographically, ids
// in range): one coalesced pass; *bad is set when a row breaks it.
template <int D>
__global__ void k_validate(const int32_t* __restrict__ T, long long nT, int nV, int* bad) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nT) return;
  int r[D];
#pragma unroll
  for (int k = 0; k < D; ++k) r[k] = T[t * D + k];
  bool ok = r[0] >= 0 && r[D - 1] < nV;
#pragma unroll
  for (int k = 1; k < D; ++k) ok = ok && r[k] > r[k - 1];
  if (t > 0) {
    bool less = false, decided = false;  // previous row < this row, lexicographically
#pragma unroll
    for (int k = 0; k < D; ++k) {
      const int q = T[(t - 1) * D + k];
      if (!decided && q != r[k]) { less = q < r[k]; decided = true; }
    }
    ok = ok && decided && less;
  }
  if (!ok) *bad = 1;
}

// I_T per vertex: first_tet[v] = first simplex whose lowest vertex is >= v (the simplices
// are sorted, so the internal simplices of any vertex range are a contiguous id range). Thread t fills
// the entries of the vertices between the previous simplex' lowest vertex and its own.
template <int D>
__global__ void k_first_tet(const int32_t* __restrict__ T, long long nT, int nV, int32_t* first_tet) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t > nT) return;
  const int a = t < nT ? T[t * D] : nV;             // the virtual simplex nT closes the array
  const int prev = t > 0 ? T[(t - 1) * D] : -1;
  for (int v = prev + 1; v <= a; ++v) first_tet[v] = (int32_t)t;
}

// simplices per second vertex (for the index of simplices grouped by second vertex, a5)
template <int D>
__global__ void k_second_count(const int32_t* __restrict__ T, long long nT, int32_t* cnt) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < nT) atomicAdd(cnt + T[t * D + 1], 1);
}
template <int D>
__global__ void k_second_fill(const int32_t* __restrict__ T, long long nT, int32_t* cursor, int32_t* perm) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < nT) perm[atomicAdd(cursor + T[t * D + 1], 1)] = (int32_t)t;
}

// ---- exclusive scan of n int32 values, in place, three launches ----------------------------------
constexpr int kScanBlock = 1024, kScanItems = 4, kScanChunk = kScanBlock * kScanItems;

__device__ __forceinline__ int block_scan_1024(int x, int* scratch, int* total) {  // exclusive, 1024 threads
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int inc = x;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int y = __shfl_up_sync(0xFFFFFFFFu, inc, d);
    if (lane >= d) inc += y;
  }
  if (lane == 31) scratch[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int w = scratch[lane];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int y = __shfl_up_sync(0xFFFFFFFFu, w, d);
      if (lane >= d) w += y;
    }
    scratch[lane] = w;
  }
  __syncthreads();
  const int base = warp ? scratch[warp - 1] : 0;
  *total = scratch[31];
  __syncthreads();
  return base + inc - x;
}

__global__ void __launch_bounds__(kScanBlock) k_scan_sums(const int32_t* __restrict__ a, long long n, int32_t* sums) {
  __shared__ int scratch[32];
  const long long base = (long long)blockIdx.x * kScanChunk + (long long)threadIdx.x * kScanItems;
  int s = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i)
    if (base + i < n) s += a[base + i];
  int tot;
  block_scan_1024(s, scratch, &tot);
  if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}
// one block: exclusive scan of the chunk sums (any count, carried serially over 1024-wide rounds)
__global__ void __launch_bounds__(kScanBlock) k_scan_top(int32_t* sums, int m) {
  __shared__ int scratch[32];
  int carry = 0;
  for (int b = 0; b < m; b += kScanBlock) {
    const int i = b + threadIdx.x;
    const int x = i < m ? sums[i] : 0;
    int tot;
    const int ex = block_scan_1024(x, scratch, &tot);
    if (i < m) sums[i] = carry + ex;
    carry += tot;
  }
}
__global__ void __launch_bounds__(kScanBlock) k_scan_apply(int32_t* a, long long n, const int32_t* __restrict__ sums) {
  __shared__ int scratch[32];
  const long long base = (long long)blockIdx.x * kScanChunk + (long long)threadIdx.x * kScanItems;
  int v[kScanItems], s = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) { v[i] = base + i < n ? a[base + i] : 0; s += v[i]; }
  int tot;
  int ex = block_scan_1024(s, scratch, &tot) + sums[blockIdx.x];
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    if (base + i < n) a[base + i] = ex;
    ex += v[i];
  }
}
// a[0..n) -> exclusive prefix sums in place (int32; the caller guarantees the total fits). scratch: >= n/4096+1 ints
inline cudaError_t exclusive_scan_i32(int32_t* a, long long n, int32_t* scratch, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  const int blocks = (int)((n + kScanChunk - 1) / kScanChunk);
  k_scan_sums<<<blocks, kScanBlock, 0, st>>>(a, n, scratch);
  k_scan_top<<<1, kScanBlock, 0, st>>>(scratch, blocks);
  k_scan_apply<<<blocks, kScanBlock, 0, st>>>(a, n, scratch);
  return cudaGetLastError();
}

// ---- tiles ---------------------------------------------------------------------------------------
// tile_of[v] for every vertex: one thread per tile writes its (<= 256) rows.
__global__ void k_tile_of(const int32_t* __restrict__ tile_vlo, const int32_t* __restrict__ tile_nrows, int nTiles,
                          int32_t* tile_of) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nTiles) return;
  const int lo = tile_vlo[i], n = tile_nrows[i];
  for (int r = 0; r < n; ++r) tile_of[lo + r] = i;
}
// internal simplices of every tile: I_T restricted to the tile's vertex range
__global__ void k_tile_internal(const int32_t* __restrict__ first_tet, const int32_t* __restrict__ tile_vlo,
                                const int32_t* __restrict__ tile_nrows, int nTiles, int32_t* t_lo, int32_t* s_int) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nTiles) return;
  const int a = first_tet[tile_vlo[i]], b = first_tet[tile_vlo[i] + tile_nrows[i]];
  t_lo[i] = a;
  s_int[i] = b - a;
}

// T_ex: simplex t is external to every tile it touches other than the tile of its lowest
// vertex. COUNT: sizes per tile; else: append t to each such tile's list (order fixed by the sort below).
template <int D, bool COUNT>
__global__ void k_external(const int32_t* __restrict__ T, long long nT, const int32_t* __restrict__ tile_of,
                           int32_t* cnt_or_cursor, int32_t* raw) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nT) return;
  const int t0 = tile_of[T[t * D]];
  int seen[D - 1], ns = 0;
#pragma unroll
  for (int k = 1; k < D; ++k) {
    const int tk = tile_of[T[t * D + k]];
    bool dup = tk == t0;
    for (int s = 0; s < ns; ++s) dup |= seen[s] == tk;
    if (dup) continue;
    seen[ns++] = tk;
    const int pos = atomicAdd(cnt_or_cursor + tk, 1);
    if (!COUNT) raw[pos] = (int32_t)t;
  }
}

// In-place bitonic sort of n2 (power of two) ints in shared memory by the whole block.
__device__ __forceinline__ void bitonic_sort_smem(int32_t* a, int n2) {
  for (int k = 2; k <= n2; k <<= 1)
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = threadIdx.x; i < n2; i += blockDim.x) {
        const int p = i ^ j;
        if (p > i) {
          const int x = a[i], y = a[p];
          const bool up = (i & k) == 0;
          if ((x > y) == up) { a[i] = y; a[p] = x; }
        }
      }
      __syncthreads();
    }
}
__host__ __device__ inline int pow2_ceil(int n) { int p = 1; while (p < n) p <<= 1; return p; }

// One block per tile: sort the tile's raw T_ex list ascending and write it to its padded place in `tex`
// (padding entries = 0). Dynamic shared memory: pow2_ceil(largest list) ints.
__global__ void k_sort_external(const int32_t* __restrict__ raw, const int32_t* __restrict__ raw_off,
                                const long long* __restrict__ tex_off, int32_t* tex) {
  extern __shared__ int32_t sh[];
  const int i = blockIdx.x;
  const int lo = raw_off[i], n = raw_off[i + 1] - lo;
  const int n2 = pow2_ceil(n < 1 ? 1 : n);
  for (int j = threadIdx.x; j < n2; j += blockDim.x) sh[j] = j < n ? raw[lo + j] : INT_MAX;
  __syncthreads();
  bitonic_sort_smem(sh, n2);
  int32_t* out = tex + tex_off[i];
  const int npad = (n + 3) & ~3;
  for (int j = threadIdx.x; j < npad; j += blockDim.x) out[j] = j < n ? sh[j] : 0;
}

// exclusive block scan for any block size that is a multiple of 32 (<= 1024); scratch: 32 ints
__device__ __forceinline__ int block_scan_any(int x, int* scratch, int* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  int inc = x;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int y = __shfl_up_sync(0xFFFFFFFFu, inc, d);
    if (lane >= d) inc += y;
  }
  if (lane == 31) scratch[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int w = lane < nw ? scratch[lane] : 0;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int y = __shfl_up_sync(0xFFFFFFFFu, w, d);
      if (lane >= d) w += y;
    }
    scratch[lane] = w;
  }
  __syncthreads();
  const int base = warp ? scratch[warp - 1] : 0;
  *total = scratch[31];
  __syncthreads();
  return base + inc - x;
}

// Per-tile inputs / outputs of the halo pass (struct of arrays, one entry per tile, all DEVICE).
struct TileArrays {
  const int32_t* vlo; const int32_t* nrows; const int32_t* t_lo; const int32_t* s_int; const int32_t* s_ext;
  const long long* tex_off; const long long* stg_off; const long long* gid_off;
  int32_t* nlo; int32_t* nhalo;   // written by the counting pass, read by the writing pass
};

__device__ __forceinline__ int lower_bound_smem(const int32_t* a, int n, int v) {
  int lo = 0, hi = n;
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (a[mid] < v) lo = mid + 1; else hi = mid;
  }
  return lo;
}

// One block per tile. The halo of a tile = the vertices outside it that share a staged simplex (internal
// range I_T + T_ex list) with it; sorted, it gives the tile-local numbering
//   [halo below the tile][the tile's vertices][halo above]   (ascending with the global id).
// WRITE = false: count only (nlo, nhalo). WRITE = true: write gid (local -> global) and loc (the staged
// simplices in local ids, LB bytes each, 4 per simplex). Dynamic shared memory: 2 * n2 ints, n2 =
// pow2_ceil(D * largest staged count); a tile with more vertex references than ref_cap raises *too_big.
template <int D, int LB, bool WRITE>
__global__ void k_halo(const int32_t* __restrict__ T, const int32_t* __restrict__ tex, TileArrays A, int ref_cap,
                       int32_t* gid, void* loc, int* too_big) {
  extern __shared__ int32_t sh[];
  __shared__ int scratch[32];
  __shared__ int s_nlo;
  const int i = blockIdx.x;
  const int vlo = A.vlo[i], nrows = A.nrows[i], vhi = vlo + nrows;
  const int t_lo = A.t_lo[i], s_int = A.s_int[i], s_ext = A.s_ext[i], S = s_int + s_ext;
  const int n = S * D;
  if (n > ref_cap) {
    if (threadIdx.x == 0) { *too_big = 1; if (!WRITE) { A.nlo[i] = 0; A.nhalo[i] = 0; } }
    return;
  }
  const int n2 = pow2_ceil(n < 1 ? 1 : n);
  int32_t* refs = sh;
  int32_t* halo = sh + n2;
  const int32_t* ex = tex + A.tex_off[i];
  for (int j = threadIdx.x; j < n2; j += blockDim.x) {
    int v = INT_MAX;
    if (j < n) {
      const int s = j / D, k = j - s * D;
      const long long t = s < s_ext ? ex[s] : t_lo + (s - s_ext);
      v = T[t * D + k];
      if (v >= vlo && v < vhi) v = INT_MAX;  // a vertex of the tile itself
    }
    refs[j] = v;
  }
  __syncthreads();
  bitonic_sort_smem(refs, n2);
  // unique: each thread owns a contiguous chunk
  const int per = (n2 + blockDim.x - 1) / blockDim.x;
  const int c0 = min(n2, (int)threadIdx.x * per), c1 = min(n2, c0 + per);
  int heads = 0;
  for (int j = c0; j < c1; ++j) heads += (refs[j] != INT_MAX && (j == 0 || refs[j] != refs[j - 1])) ? 1 : 0;
  int nhalo;
  int pos = block_scan_any(heads, scratch, &nhalo);
  for (int j = c0; j < c1; ++j)
    if (refs[j] != INT_MAX && (j == 0 || refs[j] != refs[j - 1])) halo[pos++] = refs[j];
  __syncthreads();
  if (threadIdx.x == 0) s_nlo = lower_bound_smem(halo, nhalo, vlo);
  __syncthreads();
  const int nlo = s_nlo;
  if (!WRITE) {
    if (threadIdx.x == 0) { A.nlo[i] = nlo; A.nhalo[i] = nhalo; }
    return;
  }
  const int nloc = nhalo + nrows;
  int32_t* g = gid + A.gid_off[i];
  for (int j = threadIdx.x; j < ((nloc + 3) & ~3); j += blockDim.x)
    g[j] = j >= nloc ? 0 : (j < nlo ? halo[j] : (j < nlo + nrows ? vlo + (j - nlo) : halo[j - nrows]));
  const long long so = A.stg_off[i];
  for (int s = threadIdx.x; s < ((S + 3) & ~3); s += blockDim.x) {
    uint32_t l[4] = {0u, 0u, 0u, 0u};
    if (s < S) {
      const long long t = s < s_ext ? ex[s] : t_lo + (s - s_ext);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (k >= D) { l[k] = LB == 1 ? 0xFFu : 0xFFFFu; continue; }
        const int v = T[t * D + k];
        if (v >= vlo && v < vhi) {
          l[k] = (uint32_t)(nlo + (v - vlo));
        } else {
          const int j = lower_bound_smem(halo, nhalo, v);
          l[k] = (uint32_t)(j < nlo ? j : j + nrows);
        }
      }
    }
    if constexpr (LB == 1) {
      reinterpret_cast<uint32_t*>(loc)[so + s] = l[0] | (l[1] << 8) | (l[2] << 16) | (l[3] << 24);
    } else {
      reinterpret_cast<uint2*>(loc)[so + s] = make_uint2(l[0] | (l[1] << 16), l[2] | (l[3] << 16));
    }
  }
}

// largest facet group of a vertex: D-1 facets per simplex of its run + facet 0 of every simplex whose
// second vertex it is (sizes the walk kernel's private tables)
template <int D>
__global__ void k_gmax(const int32_t* __restrict__ first_tet, const int32_t* __restrict__ opp_first, int nV, int* out) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  int g = 0;
  if (v < nV) g = (D - 1) * (first_tet[v + 1] - first_tet[v]) + (opp_first[v + 1] - opp_first[v]);
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) g = max(g, __shfl_xor_sync(0xFFFFFFFFu, g, d));
  if ((threadIdx.x & 31) == 0 && g > 0) atomicMax(out, g);
}

__global__ void k_gather(const int32_t* __restrict__ src, const int32_t* __restrict__ idx, int n, int32_t* dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = src[idx[i]];
}

}  // namespace init
}  // namespace gale
