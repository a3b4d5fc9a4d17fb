// gale_kernels.cuh — sm_100a kernels of the GALE relation hot path.
//
// One thread block owns one *tile*: a contiguous vertex sub-range [v_lo, v_lo+nrows) of a cluster
// (a tile plays the role of the paper's <=100-vertex segment; a cluster is the
// request unit). gale_mesh_create stores, per tile, the simplices incident to it
// (internal ones = rows I_T of T; external ones = the tile's T_ex list)
// re-encoded in *tile-local* 16-bit vertex ids that ascend with the global id:
//     [lower halo 0..nlo) [tile vertices nlo..nlo+nrows) [upper halo ..nloc)
// ("halo" = vertices outside the tile that share a simplex with it). The block
//   a1  stages that list (8 B per simplex), the external simplices' global ids and the halo's
//       global ids into shared memory with 16-byte cp.async,
//   a2  VT: counts incidences per row with shared-memory atomics; the atomic's return value is the
//       entry's (unordered) rank and stays in a register; after a block scan the entries are
//       scattered without atomics and each row's atomically ranked part is put in order (rows are
//       short); the simplices whose *lowest* vertex is v are the contiguous run
//       first_tet[v]..first_tet[v+1] and need neither,
//   a3  VV: one bit per (row, local neighbour) in a rows x nloc bitmap (atomicOr: "no duplicates",
//       PAPER.md:228); local ids ascend with global ids, so expanding a row yields it sorted,
//   a4  TT: facets (sorted local-id tuples packed in 32 bits) are matched in a shared-memory
//       open-addressing table; an external simplex can only meet an internal one through its
//       facet opposite its lowest vertex, and only if its second vertex is in the tile,
//   a5  TT fallback: the facet opposite the lowest vertex a of an internal simplex (a,b,..) with
//       b outside the tile may have its coface outside the staged set; a warp resolves it from
//       global memory through the run of simplices starting with b and the index of simplices
//       whose second vertex is b (DESIGN.md §TT fallback),
//   a6  writes the CSR pieces with coalesced stores (ids translated back to global).
// All arithmetic is integer index work; no floating point.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gale {

constexpr int kMaxBatch = 128;         // clusters per kernel launch (descriptor lives in kernel params)
constexpr int kItems = 8;              // staged simplices per thread (ranks live in registers)
constexpr uint32_t kEmpty32 = 0xFFFFFFFFu;
constexpr uint16_t kNoMate = 0xFFFFu;
constexpr int kMaxRec = 32766;         // facet records per tile (15-bit record ids)
constexpr int kMaxLocal4 = 1024;       // tetrahedra: 10-bit local ids (30-bit facet key)
constexpr int kMaxLocal3 = 65534;      // triangles: 16-bit local ids
constexpr int kMaxRowPart = 1023;      // atomically ranked entries of one VT row (10-bit ranks)
constexpr int kMaxNnz16 = 65535;       // VT / VV entries of one tile (16-bit packed scan)

enum { REL_VT = 1, REL_VV = 2, REL_TT = 4, MODE_COUNT = 8 };
enum { ERR_TT_TABLE_FULL = 2, ERR_SIZE_MISMATCH = 4 };

// Per-tile record built by gale_mesh_create (80 bytes, 16-byte aligned).
struct TileDesc {
  int32_t v_lo, nrows;        // vertices [v_lo, v_lo+nrows)
  int32_t t_lo, s_int;        // internal simplices [t_lo, t_lo+s_int)
  int32_t s_ext;              // external simplices (T_ex of the tile)
  int32_t nlo, nhalo;         // halo vertices below v_lo / in total
  int32_t row_rel, tt_rel;    // first row / first TT row of the tile inside its cluster
  int32_t vt_rel, vv_rel;     // first VT / VV entry of the tile inside its cluster
  int32_t vt_nnz, vv_nnz;     // entries of the tile (fixed at create; the kernel re-derives them)
  int32_t pad0;
  long long stg_off;          // first staged simplex of the tile in DeviceMesh::loc (even)
  long long tex_off;          // first entry in DeviceMesh::tex (multiple of 4)
  long long halo_off;         // first entry in DeviceMesh::halo (multiple of 4)
};
static_assert(sizeof(TileDesc) == 80, "TileDesc layout");

// Device-resident index built by gale_mesh_create (all pointers DEVICE).
struct DeviceMesh {
  const int32_t* T;                   // [nT*D] canonical simplices (caller's array)
  const int32_t* first_tet;           // [nV+1] first simplex whose lowest vertex is >= v  (I_T)
  const int32_t* opp_first;           // [nV+1] first position in opp_perm whose second vertex is >= v
  const int32_t* opp_perm;            // [nT]   simplex ids grouped by second vertex
  const TileDesc* tiles;              // [nTiles]
  const uint2* loc;                   // staged simplices in tile-local ids, 4 x uint16 each
  const int32_t* tex;                 // per-tile ascending global ids of external simplices (T_ex)
  const int32_t* halo;                // per-tile ascending global ids of halo vertices
  const int32_t* cluster_tile_begin;  // [nC+1]
  int32_t* err;                       // sticky device error flags (host-mapped)
};

// Shared-memory capacities (maxima over all tiles of the mesh, fixed at create). A field is 0 when
// the launch's relation mask does not need the region.
struct SmemCfg {
  int tv;        // rows (vertices) per tile
  int smax;      // staged simplices (even)
  int sext;      // external simplices (multiple of 4)
  int nhalo;     // halo vertices (multiple of 4)
  int W;         // bitmap words per row (odd), 0 without VV
  int cap;       // facet table slots, 0 without TT
  int nrec;      // internal facet records = 4 * max s_int, 0 without TT
  int vt_max;    // VT entries staged for write-out, 0 without VT or in count mode
  int vv_max;    // VV entries staged for write-out
};

struct SmemLayout {
  int tets, texid, halo, ft, cnt, off_vt, off_vv, bm, mate, keys, vt16, vv16, scan, total;
};

__host__ __device__ inline int align16(int x) { return (x + 15) & ~15; }

__host__ __device__ inline SmemLayout make_layout(const SmemCfg& c) {
  SmemLayout L;
  int o = 0;
  L.tets = o;   o = align16(o + c.smax * 8);
  L.texid = o;  o = align16(o + c.sext * 4);
  L.halo = o;   o = align16(o + c.nhalo * 4);
  L.ft = o;     o = align16(o + (c.tv + 1) * 4);
  L.cnt = o;    o = align16(o + c.tv * 4);
  L.off_vt = o; o = align16(o + (c.tv + 1) * 4);
  L.off_vv = o; o = align16(o + (c.tv + 1) * 4);
  L.bm = o;     o = align16(o + c.tv * c.W * 4);
  L.mate = o;   o = align16(o + c.nrec * 2);
  // the facet table is dead once every facet is inserted; the write-out staging reuses it
  L.keys = o;
  L.vt16 = o;
  L.vv16 = align16(o + c.vt_max * 2);
  const int stage_end = align16(L.vv16 + c.vv_max * 2);
  const int keys_end = align16(o + c.cap * 4);
  o = stage_end > keys_end ? stage_end : keys_end;
  L.scan = o;   o = align16(o + 40 * 4);
  L.total = o;
  return L;
}

// Per-launch batch descriptor, passed by value in kernel parameter space (no H2D copy).
struct BatchParams {
  int n_clusters;
  uint32_t mask;
  int tile_base;                     // count mode: first tile of the launch
  int total_rows;                    // VT/VV rows of the whole batch
  int total_vt_nnz, total_vv_nnz;    // terminal offsets
  int tile_prefix[kMaxBatch + 1];    // tiles of the batch before cluster slot i  (block -> cluster slot)
  int cluster[kMaxBatch];            // cluster id of slot i
  int row_base[kMaxBatch];           // first VT/VV row of slot i in the batch
  int vt_base[kMaxBatch];            // first VT index position of slot i
  int vv_base[kMaxBatch];
  int tt_base[kMaxBatch];            // first TT row of slot i
};

struct OutPtrs {
  int32_t* vt_offsets;
  int32_t* vt_indices;
  int32_t* vv_offsets;
  int32_t* vv_indices;
  int32_t* tt_indices;
  long long* stats;                  // count mode: [nTiles][4] = VT nnz, VV nnz, distinct facets, 0
};

// ------------------------------------------------------------------------------------------------
// Guard codes go to a host-mapped word (plain store: no PCIe atomics needed; any code is fatal).
__device__ __forceinline__ void raise_err(int32_t* err, int code) { *reinterpret_cast<volatile int32_t*>(err) = code; }

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

template <int D>
__device__ __forceinline__ void unpack_local(const uint2 q, int (&l)[4]) {
  l[0] = q.x & 0xFFFF; l[1] = q.x >> 16; l[2] = q.y & 0xFFFF; l[3] = q.y >> 16;
}

// Key of the facet opposite local vertex k (runtime k): ascending local ids packed in 32 bits.
template <int D>
__device__ __forceinline__ uint32_t facet_key(const int (&l)[4], int k) {
  if constexpr (D == 4) {
    const int a = k == 0 ? l[1] : l[0];
    const int b = k <= 1 ? l[2] : l[1];
    const int c = k <= 2 ? l[3] : l[2];
    return (uint32_t)a | ((uint32_t)b << 10) | ((uint32_t)c << 20);
  } else {
    const int a = k == 0 ? l[1] : l[0];
    const int b = k <= 1 ? l[2] : l[1];
    return (uint32_t)a | ((uint32_t)b << 16);
  }
}
__device__ __forceinline__ uint32_t hash_key(uint32_t key) {
  uint32_t h = key * 0x9E3779B1u;
  h ^= h >> 15;
  h *= 0x85EBCA77u;
  h ^= h >> 13;
  return h;
}

// Insert facet `key` of record `rec` (staged simplex `s`); on meeting its twin, join the two.
// Table word = (17-bit fingerprint << 15) | record. Records: 4*i+k for internal simplex i,
// 4*s_int + e for the facet opposite the lowest vertex of external simplex e.
// Returns true if the facet was new (claimed an empty slot).
template <int D>
__device__ __forceinline__ bool tt_insert(uint32_t* tbl, int cap, const uint2* tets, uint16_t* mate, int s_int,
                                          int s_ext, uint32_t key, int rec, int s, int32_t* err) {
  const uint32_t h = hash_key(key);
  const uint32_t me = ((h & 0x1FFFFu) << 15) | (uint32_t)rec;
  uint32_t slot = __umulhi(h, (uint32_t)cap);
  for (int probe = 0; probe < cap; ++probe) {
    uint32_t cur = tbl[slot];
    if (cur == kEmpty32) {
      cur = atomicCAS(&tbl[slot], kEmpty32, me);
      if (cur == kEmpty32) return true;
    }
    if ((cur ^ me) < 0x8000u) {  // same fingerprint: compare the facets themselves
      const int orec = cur & 0x7FFF;
      const bool oint = orec < 4 * s_int;
      const int os = oint ? s_ext + (orec >> 2) : orec - 4 * s_int;
      int ol[4];
      unpack_local<D>(tets[os], ol);
      if (facet_key<D>(ol, oint ? (orec & 3) : 0) == key) {
        if (oint) mate[orec] = (uint16_t)s;
        if (rec < 4 * s_int) mate[rec] = (uint16_t)os;
        return false;
      }
    }
    slot = slot + 1 == (uint32_t)cap ? 0u : slot + 1;
  }
  raise_err(err, ERR_TT_TABLE_FULL);
  return false;
}

template <int D>
__device__ __forceinline__ void load_simplex_global(const int32_t* T, int t, int (&v)[4]) {
  if constexpr (D == 4) {
    const int4 q = __ldg(reinterpret_cast<const int4*>(T) + t);
    v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
  } else {
    v[0] = __ldg(T + (long long)t * 3); v[1] = __ldg(T + (long long)t * 3 + 1); v[2] = __ldg(T + (long long)t * 3 + 2);
    v[3] = -1;
  }
}

// a5, executed by a whole warp for one request: coface != self of the facet (b, c[, d]) whose
// vertices all lie outside the tile. Both cofaces of a facet with lowest vertex b have b as
// lowest or second-lowest vertex: candidates are the run of simplices starting with b and the
// simplices whose second vertex is b; each lane tests one candidate.
template <int D>
__device__ __forceinline__ int tt_fallback_warp(const DeviceMesh& M, int b, int c, int d, int self, int lane) {
  const int f0 = __ldg(M.first_tet + b), n1 = __ldg(M.first_tet + b + 1) - f0;
  const int o0 = __ldg(M.opp_first + b), n2 = __ldg(M.opp_first + b + 1) - o0;
  for (int base = 0; base < n1 + n2; base += 32) {
    const int idx = base + lane;
    bool hit = false;
    int cand = -1;
    if (idx < n1 + n2) {
      cand = idx < n1 ? f0 + idx : __ldg(M.opp_perm + o0 + (idx - n1));
      if (cand != self) {
        int v[4];
        load_simplex_global<D>(M.T, cand, v);
        if constexpr (D == 4)
          hit = (v[1] == c || v[2] == c || v[3] == c) && (v[2] == d || v[3] == d);
        else
          hit = (v[1] == c || v[2] == c);
      }
    }
    const unsigned m = __ballot_sync(0xFFFFFFFFu, hit);
    if (m) return __shfl_sync(0xFFFFFFFFu, cand, __ffs(m) - 1);
  }
  return -1;
}

// Block-wide exclusive scan of one value per thread. Returns the exclusive prefix; *total gets
// the block sum. scratch: 33 ints of shared memory.
template <int NT>
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t x, uint32_t* scratch, uint32_t* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t inc = x;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, inc, d);
    if (lane >= d) inc += y;
  }
  if (lane == 31) scratch[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = lane < (NT / 32) ? scratch[lane] : 0u;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, w, d);
      if (lane >= d) w += y;
    }
    scratch[lane] = w;  // inclusive warp totals
  }
  __syncthreads();
  const uint32_t base = warp == 0 ? 0u : scratch[warp - 1];
  *total = scratch[NT / 32 - 1];
  return base + inc - x;
}

__device__ __forceinline__ void insertion_sort16(uint16_t* a, int n) {
  for (int i = 1; i < n; ++i) {
    const uint16_t x = a[i];
    int j = i - 1;
    while (j >= 0 && a[j] > x) {
      a[j + 1] = a[j];
      --j;
    }
    a[j + 1] = x;
  }
}

// ------------------------------------------------------------------------------------------------
// The batch kernel: VT + VV + TT for every tile of the requested clusters (or, with MODE_COUNT,
// the exact output sizes of tiles [tile_base, tile_base + gridDim.x) — the paper's leader producer
// likewise sizes its relation arrays before launch).
template <int D, int NT>
__global__ void __launch_bounds__(NT, (NT <= 256 ? 4 : 2))
gale_batch_kernel(const DeviceMesh M, const __grid_constant__ BatchParams P, const SmemCfg C, const OutPtrs O) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t mask = P.mask;
  const bool count_only = (mask & MODE_COUNT) != 0;

  // ---- block -> (cluster slot, tile) ----------------------------------------------------------
  int slot = 0, tile;
  if (count_only) {
    tile = P.tile_base + (int)blockIdx.x;
  } else {
    if (blockIdx.x == 0 && tid == 0) {  // terminal offsets (also covers batches without rows)
      if (mask & REL_VT) { O.vt_offsets[0] = 0; O.vt_offsets[P.total_rows] = P.total_vt_nnz; }
      if (mask & REL_VV) { O.vv_offsets[0] = 0; O.vv_offsets[P.total_rows] = P.total_vv_nnz; }
    }
    if ((int)blockIdx.x >= P.tile_prefix[P.n_clusters]) return;
    int lo = 0, hi = P.n_clusters;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (P.tile_prefix[mid] <= (int)blockIdx.x) lo = mid; else hi = mid;
    }
    slot = lo;
    tile = __ldg(M.cluster_tile_begin + P.cluster[slot]) + ((int)blockIdx.x - P.tile_prefix[slot]);
  }
  TileDesc td;
  {
    const int4* src = reinterpret_cast<const int4*>(M.tiles + tile);
    int4* dst = reinterpret_cast<int4*>(&td);
#pragma unroll
    for (int i = 0; i < (int)(sizeof(TileDesc) / 16); ++i) dst[i] = __ldg(src + i);
  }
  const int v_lo = td.v_lo, nrows = td.nrows, t_lo = td.t_lo, s_int = td.s_int, s_ext = td.s_ext, nlo = td.nlo;
  const int S = s_int + s_ext;
  const int W = C.W;

  const SmemLayout L = make_layout(C);
  uint2* tets = reinterpret_cast<uint2*>(smem + L.tets);
  int32_t* texid = reinterpret_cast<int32_t*>(smem + L.texid);
  int32_t* halo = reinterpret_cast<int32_t*>(smem + L.halo);
  int32_t* ft = reinterpret_cast<int32_t*>(smem + L.ft);
  uint32_t* cnt = reinterpret_cast<uint32_t*>(smem + L.cnt);
  int32_t* off_vt = reinterpret_cast<int32_t*>(smem + L.off_vt);
  int32_t* off_vv = reinterpret_cast<int32_t*>(smem + L.off_vv);
  uint32_t* bm = reinterpret_cast<uint32_t*>(smem + L.bm);
  uint16_t* mate = reinterpret_cast<uint16_t*>(smem + L.mate);
  uint32_t* keys = reinterpret_cast<uint32_t*>(smem + L.keys);
  uint16_t* vt16 = reinterpret_cast<uint16_t*>(smem + L.vt16);
  uint16_t* vv16 = reinterpret_cast<uint16_t*>(smem + L.vv16);
  uint32_t* scan = reinterpret_cast<uint32_t*>(smem + L.scan);

  // ---- a1: stage + clear ----------------------------------------------------------------------
  {
    const int4* src = reinterpret_cast<const int4*>(M.loc + td.stg_off);
    int4* dst = reinterpret_cast<int4*>(tets);
    for (int i = tid; i < (S + 1) >> 1; i += NT) cp_async16(dst + i, src + i);
    const int4* tsrc = reinterpret_cast<const int4*>(M.tex + td.tex_off);
    int4* tdst = reinterpret_cast<int4*>(texid);
    for (int i = tid; i < (s_ext + 3) >> 2; i += NT) cp_async16(tdst + i, tsrc + i);
    const int4* hsrc = reinterpret_cast<const int4*>(M.halo + td.halo_off);
    int4* hdst = reinterpret_cast<int4*>(halo);
    for (int i = tid; i < (td.nhalo + 3) >> 2; i += NT) cp_async16(hdst + i, hsrc + i);
  }
  for (int i = tid; i <= nrows; i += NT) ft[i] = __ldg(M.first_tet + v_lo + i) - t_lo;
  for (int i = tid; i < nrows; i += NT) cnt[i] = 0u;
  if (mask & REL_VV) {
    int4* z = reinterpret_cast<int4*>(bm);
    for (int i = tid; i < (nrows * W + 3) >> 2; i += NT) z[i] = make_int4(0, 0, 0, 0);
  }
  if (mask & REL_TT) {
    int4* z = reinterpret_cast<int4*>(keys);
    for (int i = tid; i < (C.cap + 3) >> 2; i += NT) z[i] = make_int4(-1, -1, -1, -1);
    int4* m4 = reinterpret_cast<int4*>(mate);
    for (int i = tid; i < (s_int + 1) >> 1; i += NT) m4[i] = make_int4(-1, -1, -1, -1);
  }
  if (tid == 0) scan[36] = 0u;  // distinct facets (count mode)
  cp_async_wait_all();
  __syncthreads();

  // ---- pass A: VT counts (ranks stay in registers), VV bitmap, facet matching -----------------
  uint32_t rk[kItems];
#pragma unroll
  for (int j = 0; j < kItems; ++j) {
    rk[j] = 0u;
    const int s = tid + j * NT;
    if ((mask & REL_VT) && s < S) {
      int l[4];
      unpack_local<D>(tets[s], l);
      uint32_t pk = 0u;
#pragma unroll
      for (int k = 1; k < D; ++k) {
        const int r = l[k] - nlo;
        if ((unsigned)r < (unsigned)nrows) pk |= atomicAdd(&cnt[r], 1u) << (10 * (k - 1));
      }
      rk[j] = pk;
    }
  }
  if (mask & (REL_VV | REL_TT)) {
    int nnew = 0;
    for (int s = tid; s < S; s += NT) {
      int l[4];
      unpack_local<D>(tets[s], l);
      bool in[D];
#pragma unroll
      for (int k = 0; k < D; ++k) in[k] = (unsigned)(l[k] - nlo) < (unsigned)nrows;
      if (mask & REL_VV) {
        uint32_t w[D], b[D];
#pragma unroll
        for (int k = 0; k < D; ++k) { w[k] = (uint32_t)l[k] >> 5; b[k] = 1u << (l[k] & 31); }
#pragma unroll
        for (int k = 0; k < D; ++k) {
          if (!in[k]) continue;
          uint32_t* row = bm + (l[k] - nlo) * W;
#pragma unroll
          for (int j = 0; j < D; ++j)
            if (j != k) atomicOr(row + w[j], b[j]);
        }
      }
      if (mask & REL_TT) {
        if (s >= s_ext) {
          const int i = s - s_ext;
#pragma unroll
          for (int k = 0; k < D; ++k)
            nnew += tt_insert<D>(keys, C.cap, tets, mate, s_int, s_ext, facet_key<D>(l, k), 4 * i + k, s, M.err);
        } else if (in[1]) {
          nnew += tt_insert<D>(keys, C.cap, tets, mate, s_int, s_ext, facet_key<D>(l, 0), 4 * s_int + s, s, M.err);
        }
      }
    }
    if (count_only && nnew) atomicAdd(&scan[36], (uint32_t)nnew);
  }
  __syncthreads();

  // ---- row degrees -> offsets (VT in the low, VV in the high 16 bits of one scan) -------------
  uint32_t tot;
  {
    uint32_t dvt = 0, dvv = 0;
    if (tid < nrows) {
      if (mask & REL_VT) dvt = cnt[tid] + (uint32_t)(ft[tid + 1] - ft[tid]);
      if (mask & REL_VV) {
        const uint32_t* row = bm + tid * W;
        for (int w = 0; w < W; ++w) dvv += __popc(row[w]);
      }
    }
    const uint32_t ex = block_exclusive_scan<NT>(dvt | (dvv << 16), scan, &tot);
    if (tid < nrows) {
      off_vt[tid] = (int)(ex & 0xFFFFu);
      off_vv[tid] = (int)(ex >> 16);
      // from here on ft[r] = position of the first lowest-vertex entry of row r minus its simplex index
      ft[tid] = (int)(ex & 0xFFFFu) + (int)cnt[tid] - ft[tid];
    }
    if (tid == 0) { off_vt[nrows] = (int)(tot & 0xFFFFu); off_vv[nrows] = (int)(tot >> 16); }
  }
  const int n_vt = (int)(tot & 0xFFFFu), n_vv = (int)(tot >> 16);
  if (count_only) {
    __syncthreads();
    if (tid == 0) {
      O.stats[(long long)tile * 4 + 0] = n_vt;
      O.stats[(long long)tile * 4 + 1] = n_vv;
      O.stats[(long long)tile * 4 + 2] = scan[36];
      O.stats[(long long)tile * 4 + 3] = 0;
    }
    return;
  }
  if (tid == 0 && (((mask & REL_VT) && n_vt != td.vt_nnz) || ((mask & REL_VV) && n_vv != td.vv_nnz)))
    raise_err(M.err, ERR_SIZE_MISMATCH);  // the sizes fixed at create must be reproduced exactly
  const int row0 = P.row_base[slot] + td.row_rel;
  const int vt0 = P.vt_base[slot] + td.vt_rel;
  const int vv0 = P.vv_base[slot] + td.vv_rel;
  const int tt0 = P.tt_base[slot] + td.tt_rel;
  __syncthreads();
  if (tid <= nrows) {
    if (mask & REL_VT) O.vt_offsets[row0 + tid] = vt0 + off_vt[tid];
    if (mask & REL_VV) O.vv_offsets[row0 + tid] = vv0 + off_vv[tid];
  }

  // ---- pass B: scatter VT (no atomics: rank from pass A) --------------------------------------
  if (mask & REL_VT) {
#pragma unroll
    for (int j = 0; j < kItems; ++j) {
      const int s = tid + j * NT;
      if (s < S) {
        int l[4];
        unpack_local<D>(tets[s], l);
#pragma unroll
        for (int k = 1; k < D; ++k) {
          const int r = l[k] - nlo;
          if ((unsigned)r < (unsigned)nrows) vt16[off_vt[r] + (int)((rk[j] >> (10 * (k - 1))) & 1023u)] = (uint16_t)s;
        }
        if (s >= s_ext) vt16[ft[l[0] - nlo] + (s - s_ext)] = (uint16_t)s;
      }
    }
  }
  __syncthreads();

  // ---- pass C: order the ranked part of each VT row, expand the VV bitmap, emit TT ------------
  if (tid < nrows) {
    if (mask & REL_VT) insertion_sort16(vt16 + off_vt[tid], (int)cnt[tid]);
    if (mask & REL_VV) {
      const uint32_t* row = bm + tid * W;
      int p = off_vv[tid];
      for (int w = 0; w < W; ++w) {
        uint32_t bits = row[w];
        while (bits) {
          const int b = __ffs(bits) - 1;
          bits &= bits - 1;
          vv16[p++] = (uint16_t)(w * 32 + b);
        }
      }
    }
  }
  if (mask & REL_TT) {
    for (int base = tid - lane; base < s_int; base += NT) {  // warp-uniform trip count
      const int i = base + lane;
      const bool valid = i < s_int;
      int l[4] = {0, 0, 0, 0};
      int nb[4] = {-1, -1, -1, -1};
      bool need_fb = false;
      if (valid) {
        unpack_local<D>(tets[s_ext + i], l);
        const uint2 m2 = reinterpret_cast<const uint2*>(mate)[i];
        const uint32_t m[4] = {m2.x & 0xFFFFu, m2.x >> 16, m2.y & 0xFFFFu, m2.y >> 16};
#pragma unroll
        for (int k = 0; k < D; ++k)
          if (m[k] != kNoMate) nb[k] = (int)m[k] < s_ext ? texid[m[k]] : t_lo + ((int)m[k] - s_ext);
        need_fb = m[0] == kNoMate && (l[1] - nlo) >= nrows;
      }
      unsigned fbm = __ballot_sync(0xFFFFFFFFu, need_fb);
      if (fbm) {  // a5: facets with no vertex in the tile
        const int g1 = need_fb ? halo[l[1] - nrows] : 0;
        const int g2 = need_fb ? halo[l[2] - nrows] : 0;
        const int g3 = (D == 4 && need_fb) ? halo[l[3] - nrows] : 0;
        while (fbm) {
          const int src = __ffs(fbm) - 1;
          fbm &= fbm - 1;
          const int b = __shfl_sync(0xFFFFFFFFu, g1, src), c = __shfl_sync(0xFFFFFFFFu, g2, src);
          const int d = __shfl_sync(0xFFFFFFFFu, g3, src);
          const int r = tt_fallback_warp<D>(M, b, c, d, t_lo + base + src, lane);
          if (lane == src) nb[0] = r;
        }
      }
      if (valid) {
        if constexpr (D == 4) {
          reinterpret_cast<int4*>(O.tt_indices)[tt0 + i] = make_int4(nb[0], nb[1], nb[2], nb[3]);
        } else {
          int32_t* o = O.tt_indices + (long long)(tt0 + i) * 3;
          o[0] = nb[0]; o[1] = nb[1]; o[2] = nb[2];
        }
      }
    }
  }
  __syncthreads();

  // ---- a6: coalesced write-out, local ids back to global --------------------------------------
  if (mask & REL_VT) {
    for (int i = tid; i < n_vt; i += NT) {
      const int s = vt16[i];
      O.vt_indices[vt0 + i] = s < s_ext ? texid[s] : t_lo + (s - s_ext);
    }
  }
  if (mask & REL_VV) {
    for (int i = tid; i < n_vv; i += NT) {
      const int l = vv16[i];
      const int r = l - nlo;
      O.vv_indices[vv0 + i] = r < 0 ? halo[l] : (r < nrows ? v_lo + r : halo[l - nrows]);
    }
  }
}

}  // namespace gale
