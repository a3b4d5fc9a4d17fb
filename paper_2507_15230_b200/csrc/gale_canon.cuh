// gale_canon.cuh — canonical form of a simplex list on the device (SURVEY.md §8(f)-1 "canonicalisation itself").
//
// The hot path expects every row of T ascending (C1) and the rows in ascending lexicographic order (C2,
// DESIGN.md §2 reading 2): the paper's interval array I_T needs the simplices grouped by the segment of their
// lowest vertex. gale_canonicalize produces that form from any vertex order inside the
// rows and any row order:
//   1. k_sort_rows: one thread per simplex sorts its D vertex ids (a fixed network), checks their range and
//      that they are distinct, and starts the permutation perm[i] = i;
//   2. a least-significant-digit radix sort of the rows, last column first, 8 bits per pass, ceil(bits(nV-1)/8)
//      passes per column. A pass is count -> scan -> scatter over contiguous SEGMENTS of kSeg rows, one warp
//      per segment: the warp keeps 256 counters in shared memory; the counts of all (digit, segment) pairs are
//      scanned digit-major (gale_init's three-launch scan), which gives every segment the first output
//      position of each of its digits; the scatter walks the segment in order, 32 rows at a time, and ranks
//      equal digits inside the 32 with MATCH.ANY, so every pass is stable and the sort as a whole is stable
//      (equal rows keep their input order, perm is unique).
// Whole rows travel with their permutation entry, so every read is a coalesced stream; only the scatter's
// writes are scattered (16-byte rows).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gale_init.cuh"

namespace gale {
namespace canon {

constexpr int kSeg = 2048;       // rows per segment (one warp)
constexpr int kWarps = 4;        // warps (segments) per block
constexpr int kDigits = 256;

template <int D>
__device__ __forceinline__ void load_row(const int32_t* __restrict__ T, long long i, int (&v)[4]) {
  if constexpr (D == 4) {
    const int4 q = __ldg(reinterpret_cast<const int4*>(T) + i);
    v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
  } else {
    v[0] = __ldg(T + i * 3); v[1] = __ldg(T + i * 3 + 1); v[2] = __ldg(T + i * 3 + 2); v[3] = 0;
  }
}
template <int D>
__device__ __forceinline__ void store_row(int32_t* T, long long i, const int (&v)[4]) {
  if constexpr (D == 4) {
    reinterpret_cast<int4*>(T)[i] = make_int4(v[0], v[1], v[2], v[3]);
  } else {
    T[i * 3] = v[0]; T[i * 3 + 1] = v[1]; T[i * 3 + 2] = v[2];
  }
}

__device__ __forceinline__ void cswap(int& a, int& b) {
  const int lo = min(a, b), hi = max(a, b);
  a = lo; b = hi;
}

// rows ascending; bad[0] is set when an id lies outside [0, nV) or a row repeats a vertex
template <int D>
__global__ void k_sort_rows(const int32_t* __restrict__ in, long long n, int nV, int32_t* out, int32_t* perm, int* bad) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int v[4];
  load_row<D>(in, i, v);
  if constexpr (D == 4) {
    cswap(v[0], v[1]); cswap(v[2], v[3]); cswap(v[0], v[2]); cswap(v[1], v[3]); cswap(v[1], v[2]);
  } else {
    cswap(v[0], v[1]); cswap(v[1], v[2]); cswap(v[0], v[1]);
  }
  bool ok = v[0] >= 0 && v[D - 1] < nV;
#pragma unroll
  for (int k = 1; k < D; ++k) ok = ok && v[k - 1] < v[k];
  if (!ok) *bad = 1;
  store_row<D>(out, i, v);
  perm[i] = (int32_t)i;
}

// counts[d * nseg + seg] = rows of segment seg whose digit (column col, bits [shift, shift + 8)) is d
template <int D>
__global__ void __launch_bounds__(kWarps * 32) k_count(const int32_t* __restrict__ T, long long n, int col, int shift,
                                                       int nseg, int32_t* counts) {
  __shared__ int32_t hist[kWarps][kDigits];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int seg = blockIdx.x * kWarps + warp;
  for (int d = lane; d < kDigits; d += 32) hist[warp][d] = 0;
  __syncwarp();
  if (seg < nseg) {
    const long long r0 = (long long)seg * kSeg, r1 = min(r0 + kSeg, n);
    for (long long i = r0 + lane; i < r1; i += 32) {
      const int key = __ldg(T + i * D + col);
      atomicAdd(&hist[warp][(key >> shift) & (kDigits - 1)], 1);
    }
    __syncwarp();
    for (int d = lane; d < kDigits; d += 32) counts[(long long)d * nseg + seg] = hist[warp][d];
  }
}

// stable scatter of one pass: rows (and their permutation entries) of segment seg go to the positions the
// scanned counts assign to its digits, in segment order
template <int D>
__global__ void __launch_bounds__(kWarps * 32) k_scatter(const int32_t* __restrict__ T, const int32_t* __restrict__ perm, long long n,
                                                         int col, int shift, int nseg, const int32_t* __restrict__ base,
                                                         int32_t* T_out, int32_t* perm_out) {
  __shared__ int32_t next[kWarps][kDigits];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int seg = blockIdx.x * kWarps + warp;
  if (seg >= nseg) return;
  for (int d = lane; d < kDigits; d += 32) next[warp][d] = __ldg(base + (long long)d * nseg + seg);
  __syncwarp();
  const long long r0 = (long long)seg * kSeg, r1 = min(r0 + kSeg, n);
  const uint32_t lt = (1u << lane) - 1u;
  for (long long c = r0; c < r1; c += 32) {
    const long long i = c + lane;
    const bool live = i < r1;
    int v[4] = {0, 0, 0, 0};
    int32_t pi = 0;
    if (live) { load_row<D>(T, i, v); pi = __ldg(perm + i); }
    const int key = col == 0 ? v[0] : (col == 1 ? v[1] : (col == 2 ? v[2] : v[3]));
    // rows past the end get a digit of their own so that they join no group
    const uint32_t d = live ? (uint32_t)((key >> shift) & (kDigits - 1)) : (uint32_t)(kDigits + lane);
    const uint32_t m = __match_any_sync(0xFFFFFFFFu, d);
    const int leader = __ffs(m) - 1;
    int first = 0;
    if (live && lane == leader) { first = next[warp][d]; next[warp][d] = first + __popc(m); }
    first = __shfl_sync(0xFFFFFFFFu, first, leader);
    if (live) {
      const long long dst = (long long)first + __popc(m & lt);
      store_row<D>(T_out, dst, v);
      perm_out[dst] = pi;
    }
    __syncwarp();
  }
}

struct Buffers {
  int32_t* T[2];      // ping-pong row buffers, T[0] is the caller's output array
  int32_t* perm[2];   // ping-pong permutation buffers, perm[0] is the caller's (or a temporary)
  int32_t* counts;    // [256 * nseg]
  int32_t* scratch;   // scan scratch, >= 256 * nseg / 4096 + 2 ints
  int* bad;
};

inline int passes_per_column(int nV) {
  int bits = 1;
  while (bits < 31 && (1ll << bits) < (long long)nV) ++bits;
  return (bits + 7) / 8;
}

// Enqueues the whole sort on `st`; the canonical rows end in B.T[0], the permutation in B.perm[0].
template <int D>
inline cudaError_t canonicalize(const int32_t* d_in, long long n, int nV, const Buffers& B, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  const int ppc = passes_per_column(nV), total = ppc * D;
  const int nseg = (int)((n + kSeg - 1) / kSeg);
  int cur = total & 1;  // an even number of passes starts (and ends) in buffer 0
  k_sort_rows<D><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_in, n, nV, B.T[cur], B.perm[cur], B.bad);
  const unsigned blocks = (unsigned)((nseg + kWarps - 1) / kWarps);
  for (int col = D - 1; col >= 0; --col)
    for (int p = 0; p < ppc; ++p) {
      const int shift = 8 * p;
      k_count<D><<<blocks, kWarps * 32, 0, st>>>(B.T[cur], n, col, shift, nseg, B.counts);
      cudaError_t e = gale::init::exclusive_scan_i32(B.counts, (long long)kDigits * nseg, B.scratch, st);
      if (e != cudaSuccess) return e;
      k_scatter<D><<<blocks, kWarps * 32, 0, st>>>(B.T[cur], B.perm[cur], n, col, shift, nseg, B.counts, B.T[cur ^ 1], B.perm[cur ^ 1]);
      cur ^= 1;
    }
  return cudaGetLastError();
}

}  // namespace canon
}  // namespace gale
