// gale_kernels.cuh — sm_100a kernels of the GALE relation hot path.
//
// One thread block owns one *tile*: a contiguous vertex sub-range [v_lo, v_lo+nrows) of a cluster
// (a tile plays the role of the paper's <=100-vertex segment; a cluster is the
// request unit). gale_mesh_create stores, per tile, the simplices incident to it
// (internal ones = rows I_T of T; external ones = the tile's T_ex list)
// re-encoded in *tile-local* vertex ids (8-bit when no tile of the mesh has more than 255 local
// vertices, template argument LB = 1, else 16-bit) that ascend with the global id:
//     [lower halo 0..nlo) [tile vertices nlo..nlo+nrows) [upper halo ..nloc)
// ("halo" = vertices outside the tile that share a simplex with it), external simplices first.
// Every external simplex has a smaller global id than every internal one (its lowest vertex lies
// below the tile), so the staged order s = 0..S-1 ascends with the global simplex id.
//
// Kernel v7. Every per-simplex step is one thread per *staged simplex* (uniform work per lane, no
// per-vertex serial walks); only the two short per-row steps (prefix counts, VV expansion) are one
// thread per tile vertex. Phases:
//   P0  one thread arms an mbarrier and issues TMA bulk copies (cp.async.bulk) of the staged list, the
//       external simplices' global ids (T_ex) and the local->global vertex table; the others clear the
//       bitmaps / tables and read the tile's slice of the interval array I_T (first_tet);
//   P1  per staged simplex: VT incidence bit (row v, column s) for every tile vertex v of s other than
//       its lowest vertex (the simplices whose *lowest* vertex is v are the contiguous run
//       first_tet[v]..first_tet[v+1] and need no bits), and the VV bits (row v, column u) for every
//       other vertex u of s — shared-memory atomicOr is the paper's de-duplicating atomicPush
//       (Alg. 2; "no duplicates", :228) in one instruction;
//   P2  per tile vertex: prefix popcounts of its VT bitmap row, degrees, block scan -> VT / VV
//       offsets, facet-table offsets;
//   P3  per tile vertex: VV row -> ascending global ids into the VV staging area (local ids ascend
//       with global ids); then, per staged simplex (warps take 32-simplex chunks dynamically): the
//       rank of s in row v = prefix count + popc(bits below s) places its global id in the VT staging
//       area — rows come out sorted with no sort and no walk; TT facet records go into per-vertex
//       open-addressing tables with one atomicCAS: a facet whose lowest vertex is p has both cofaces
//       among run(p) and the simplices whose second vertex is p, so the second arrival of a key reads
//       the first (the table word carries key, staged index and facet number) and writes both TT
//       entries;
//   P4  VT / VV staging areas leave with TMA bulk stores (cp.async.bulk shared -> global); TT rows are
//       translated to global ids and written with 16-byte stores. The facet opposite the lowest
//       vertex a of an internal simplex (a, b, ..) with b outside the tile belongs to no vertex of this
//       tile: if b lies in the same cluster, the tile that owns b has this simplex in its T_ex list,
//       matches the facet there and writes that one TT entry (this tile then leaves it alone);
//       otherwise (cross-cluster facet) it is resolved from global memory (a5): first the run of
//       simplices starting with b, else the index of simplices whose second vertex is b.
// All arithmetic is integer index work; no floating point.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gale {

constexpr int kMaxBatch = 128;         // clusters per kernel launch (descriptor lives in kernel params)
constexpr uint32_t kEmpty32 = 0xFFFFFFFFu;
constexpr int kMaxStaged4 = 4094;      // tetrahedra: 12-bit staged index in a table word
constexpr int kMaxStaged3 = 16382;     // triangles: 14-bit staged index
constexpr int kMaxLocal4 = 512;        // tetrahedra: 9-bit local ids (18-bit facet key)
constexpr int kMaxLocal3 = 65534;      // triangles: 16-bit local ids
constexpr int kMaxNnz16 = 65535;       // VT / VV entries of one tile (16-bit packed scans)
constexpr int kMaxTileVertices = 256;

enum { REL_VT = 1, REL_VV = 2, REL_TT = 4, MODE_COUNT = 8 };
enum { ERR_TT_TABLE_FULL = 2, ERR_SIZE_MISMATCH = 4, ERR_BOUNDS = 8 };

// Per-tile record built by gale_mesh_create (80 bytes, 16-byte aligned).
struct TileDesc {
  int32_t v_lo, nrows;        // vertices [v_lo, v_lo+nrows)
  int32_t t_lo, s_int;        // internal simplices [t_lo, t_lo+s_int)
  int32_t s_ext;              // external simplices (T_ex of the tile)
  int32_t nlo, nloc;          // halo vertices below v_lo / local ids in total (halo + rows)
  int32_t row_rel, tt_rel;    // first row / first TT row of the tile inside its cluster
  int32_t vt_rel, vv_rel;     // first VT / VV entry of the tile inside its cluster
  int32_t vt_nnz, vv_nnz;     // entries of the tile (fixed at create; the kernel re-derives them)
  int32_t c_rows;             // vertices of the tile's cluster (its range is [v_lo - row_rel, .. + c_rows))
  long long stg_off;          // first staged simplex of the tile in DeviceMesh::loc (multiple of 4)
  long long tex_off;          // first entry in DeviceMesh::tex (multiple of 4)
  long long gid_off;          // first entry in DeviceMesh::gid (multiple of 4)
};
static_assert(sizeof(TileDesc) == 80, "TileDesc layout");

// What one warp works out for the block and leaves in shared memory: the tile's record and where its
// rows / entries go in the batch's output arrays.
struct BlockCtx {
  TileDesc td;
  int32_t row0, vt0, vv0, tt0, tt_slot, tile, pad0, pad1;
};
static_assert(sizeof(BlockCtx) == 112, "BlockCtx layout");

// Device-resident index built by gale_mesh_create (all pointers DEVICE).
struct DeviceMesh {
  const int32_t* T;                   // [nT*D] canonical simplices (caller's array)
  const int32_t* first_tet;           // [nV+1] first simplex whose lowest vertex is >= v  (I_T)
  const int32_t* opp_first;           // [nV+1] first position in opp_perm whose second vertex is >= v
  const int32_t* opp_perm;            // [nT]   simplex ids grouped by second vertex
  const TileDesc* tiles;              // [nTiles]
  const void* loc;                    // staged simplices in tile-local ids: 4 x uint16 each, or 4 x uint8
                                      //   when no tile of the mesh has more than 255 local vertices (SmemCfg::lb)
  const int32_t* tex;                 // per-tile ascending global ids of external simplices (T_ex)
  const int32_t* gid;                 // per-tile global vertex id of every local id (ascending)
  const int32_t* cluster_tile_begin;  // [nC+1]
  int32_t* err;                       // sticky device error flags (host-mapped)
};

// Shared-memory capacities (maxima over all tiles of the mesh, fixed at create). A field is 0 when
// the launch's relation mask does not need the region.
struct SmemCfg {
  int tv;        // rows (vertices) per tile, <= NT
  int smax;      // staged simplices (multiple of 4)
  int lb;        // bytes per local vertex id in the staged list: 1 or 2
  int sext;      // external simplices (multiple of 4)
  int nloc;      // local vertex ids (multiple of 4)
  int sint;      // internal simplices (even): fallback queue, 0 without TT
  int tbl;       // facet-table slots of a tile = VT entries + (D-2) * internal simplices, 0 without TT
  int hs;        // walk kernel only: table slots per tile vertex (even), 0 without TT
  int stage_t;   // dense kernel: 1 = stage from T + T_ex and map global -> local ids in the kernel (A/B)
  int WT;        // VT bitmap words per row (odd)
  int WV;        // VV bitmap words per row (odd), 0 without VV
  int vt_max;    // VT entries staged for write-out, 0 without VT or in count mode
  int vv_max;    // VV entries staged for write-out, 0 without VV or in count mode
};

// Byte offsets of the shared-memory regions, computed on the host (make_layout) and passed as a
// kernel parameter.
struct SmemLayout {
  int mbar, ctx, tets, texid, gid, ft, offT, offV, runpos, tbo, scan, misc;
  int bmT, bmV, dflag, zero_end;   // cleared to 0
  int pfx;
  int tbl, ttres, ones_end; // cleared to all-ones (empty table word, "no neighbour" = -1)
  int st_vt, st_vv, fbq;
  int total;
};

__host__ __device__ inline int align16(int x) { return (x + 15) & ~15; }

template <int D>
__host__ __device__ inline SmemLayout make_layout(const SmemCfg& c) {
  SmemLayout L;
  int o = 0;
  L.mbar = o;   o = align16(o + 8);
  L.ctx = o;    o = align16(o + 112);
  L.tets = o;   o = align16(o + c.smax * 4 * c.lb);
  L.texid = o;  o = align16(o + c.sext * 4);
  L.gid = o;    o = align16(o + c.nloc * 4);
  L.ft = o;     o = align16(o + (c.tv + 1) * 4);
  L.offT = o;   o = align16(o + (c.tv + 1) * 4);
  L.offV = o;   o = align16(o + (c.tv + 1) * 4);
  L.runpos = o; o = align16(o + c.tv * 4);
  L.tbo = o;    o = align16(o + (c.tv + 1) * 4);
  L.scan = o;   o = align16(o + 40 * 4);
  L.misc = o;   o = align16(o + 16);
  L.bmT = o;    o = align16(o + c.tv * c.WT * 4);
  L.bmV = o;    o = align16(o + c.tv * c.WV * 4);
  L.dflag = o;  o = align16(o + (c.tbl ? c.sext : 0));
  L.zero_end = o;
  L.pfx = o;    o = align16(o + c.tv * c.WT * 2);
  {
    // The VT / VV staging areas are written after the facet tables are dead (P3b): with TT they share
    // the tables' bytes (the region is as large as the larger of the two uses).
    const int b_vt = align16(c.vt_max ? (c.vt_max + 4) * 4 : 0), b_vv = align16(c.vv_max ? (c.vv_max + 4) * 4 : 0);
    const int b_tbl = align16(c.tbl * 4);
    L.tbl = o;
    L.st_vt = o;
    L.st_vv = o + b_vt;
    o += b_tbl > b_vt + b_vv ? b_tbl : b_vt + b_vv;
  }
  L.ttres = o;  o = align16(o + (c.tbl ? (c.sext + c.sint * D) * 4 : 0));
  L.ones_end = o;
  L.fbq = o;    o = align16(o + c.sint * 2);
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
  int uniform_tiles;                 // > 0: every cluster of the batch has this many tiles (slot = block / it)
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
  long long* stats;                  // count mode: [nTiles][4] = VT nnz, VV nnz, 0, 0
};

// Bounds-checked build (-DGALE_CHECK_BOUNDS=1, libgale_checked.so; tests/test_gpu_bounds.py): every tile
// is checked against the launch's shared-memory capacities and every computed staging index before it
// is written; a violation raises ERR_BOUNDS through the device error word and skips the write.
// compute-sanitizer is not available on the build pool, this is its stand-in. Off by default: no code.
__device__ __forceinline__ void raise_err(int32_t* err, int code);
// Output stores: the CSR arrays are written once and never read by the kernels, so plain stores are
// marked evict-first (st.global.cs) and leave L2 to the data the fall-back look-ups re-read.
#ifndef GALE_STREAM_OUT
#define GALE_STREAM_OUT 1
#endif
#if GALE_STREAM_OUT
#define GALE_ST(ptr, val) __stcs((ptr), (val))
#else
#define GALE_ST(ptr, val) (*(ptr) = (val))
#endif

#ifndef GALE_CHECK_BOUNDS
#define GALE_CHECK_BOUNDS 0
#endif
#if GALE_CHECK_BOUNDS
#define GALE_IN_BOUNDS(err, cond) ((cond) ? true : (raise_err((err), ERR_BOUNDS), false))
#else
#define GALE_IN_BOUNDS(err, cond) true
#endif

// ------------------------------------------------------------------------------------------------
// Guard codes go to a host-mapped word (plain store: no PCIe atomics needed; any code is fatal).
__device__ __forceinline__ void raise_err(int32_t* err, int code) { *reinterpret_cast<volatile int32_t*>(err) = code; }

// ---- TMA bulk copies (cp.async.bulk; SASS: UBLKCP) and their mbarrier -----------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(void* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!ok);
}
// global -> shared, completion counted in bytes on the mbarrier. 16-byte aligned, size multiple of 16.
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, void* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
// shared -> global (bulk async group of the issuing thread)
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read_all() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

// atomicOr without return value on a 32-bit shared-window address, predicated instead of branched
// (SASS: @P ATOMS.OR RZ): lanes whose vertex lies outside the tile skip it without a divergent region.
__device__ __forceinline__ void red_or_shared_if(bool p, uint32_t saddr, uint32_t v) {
  asm volatile("{\n .reg .pred q;\n setp.ne.u32 q, %0, 0;\n @q red.shared.or.b32 [%1], %2;\n}" ::"r"((uint32_t)p), "r"(saddr), "r"(v) : "memory");
}

__device__ __forceinline__ void st_shared_if(bool p, uint32_t saddr, int32_t v) {
  asm volatile("{\n .reg .pred q;\n setp.ne.u32 q, %0, 0;\n @q st.shared.b32 [%1], %2;\n}" ::"r"((uint32_t)p), "r"(saddr), "r"(v) : "memory");
}

// Local vertex ids of staged simplex s (LB bytes each).
template <int LB>
__device__ __forceinline__ void load_local(const unsigned char* tets, int s, int (&l)[4]) {
  if constexpr (LB == 2) {
    const uint2 q = reinterpret_cast<const uint2*>(tets)[s];
    l[0] = q.x & 0xFFFF; l[1] = q.x >> 16; l[2] = q.y & 0xFFFF; l[3] = q.y >> 16;
  } else {
    const uint32_t q = reinterpret_cast<const uint32_t*>(tets)[s];
    l[0] = q & 0xFF; l[1] = (q >> 8) & 0xFF; l[2] = (q >> 16) & 0xFF; l[3] = q >> 24;
  }
}

// a5, one request per thread: coface != self of the facet (b, c[, d]) (ascending global ids) whose
// vertices all lie outside the requesting cluster. Both cofaces of a facet with lowest vertex b have b as
// lowest or second-lowest vertex: candidates are the run [f0, f1) of simplices starting with b (I_T,
// PAPER.md:178) and the simplices whose second vertex is b (those are (x, b, c, d) exactly). Candidates
// are fetched four at a time without early exit so that their loads overlap.
template <int D>
__device__ __forceinline__ int tt_fallback(const DeviceMesh& M, int f0, int f1, int b, int c, int d, int self) {
  int found = -1;
  if constexpr (D == 4) {
    const int4* T4 = reinterpret_cast<const int4*>(M.T);
    for (int t = f0; t < f1; t += 4) {
      int4 q[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) q[u] = __ldg(T4 + min(t + u, f1 - 1));
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const bool hit = (q[u].y == c && (q[u].z == d || q[u].w == d)) || (q[u].z == c && q[u].w == d);
        if (hit) found = min(t + u, f1 - 1);
      }
    }
    if (found >= 0) return found;  // measured: > 99 % of the cofaces start with b
    const int o0 = __ldg(M.opp_first + b), o1 = __ldg(M.opp_first + b + 1);
    for (int j = o0; j < o1; j += 4) {
      int t[4];
      int4 q[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) t[u] = __ldg(M.opp_perm + min(j + u, o1 - 1));
#pragma unroll
      for (int u = 0; u < 4; ++u) q[u] = __ldg(T4 + t[u]);
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (t[u] != self && q[u].z == c && q[u].w == d) found = t[u];
    }
  } else {
    for (int t = f0; t < f1; ++t) {
      const int v1 = __ldg(M.T + (long long)t * 3 + 1), v2 = __ldg(M.T + (long long)t * 3 + 2);
      if (v1 == c || v2 == c) found = t;
    }
    if (found >= 0) return found;
    const int o0 = __ldg(M.opp_first + b), o1 = __ldg(M.opp_first + b + 1);
    for (int j = o0; j < o1; ++j) {
      const int t = __ldg(M.opp_perm + j);
      if (t != self && __ldg(M.T + (long long)t * 3 + 2) == c) found = t;
    }
  }
  return found;
}

// Block-wide exclusive scan of one value per thread. Returns the exclusive prefix; *total gets
// the block sum. scratch: 33 ints of shared memory. Ends with all threads past the last barrier.
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

// ------------------------------------------------------------------------------------------------
// TT tables. A table word of vertex p's group = key | s << kKeyBits | k << 30: the facet's
// vertices other than p (local ids, ascending), the staged simplex s it belongs to, and the local
// vertex k it is opposite to. Vertex p's table has as many slots as p has VT entries not in its own
// run plus D-1 per simplex of its run — an upper bound of its records (the simplices whose second
// vertex is p are among the former), so a table cannot fill up; with every interior facet recorded
// twice the usual load is about one third.
template <int D>
struct FacetBits {
  static constexpr int kKeyBits = D == 4 ? 18 : 16;
  static constexpr uint32_t kKeyMask = (1u << kKeyBits) - 1u;
  static constexpr uint32_t kIdxMask = (1u << (30 - kKeyBits)) - 1u;
};

// Where the TT results of a tile live in shared memory, as GLOBAL simplex ids (-1 = none):
//   [entry 0 of every external simplex: xpad words][D entries of every internal simplex]
struct TTRes {
  int32_t* res;
  const int32_t* texid;
  int s_ext, xpad, t_lo;
  int cap;  // words (bounds-checked build)
};

// Place facet k of staged simplex s with key `key` in the table [tbl, tbl+m): claim an empty slot, or
// meet the record that holds the same key (the other coface) and write both TT entries.
template <int D>
__device__ __forceinline__ void facet_place(uint32_t* tbl, uint32_t m, uint32_t key, int s, int k, const TTRes& R,
                                            int s_all, int32_t* err) {
  using FB = FacetBits<D>;
  if (!GALE_IN_BOUNDS(err, m > 0 && (uint32_t)s <= FB::kIdxMask && key <= FB::kKeyMask && k >= 0 && k < D && s < s_all)) return;
  const uint32_t word = key | ((uint32_t)s << FB::kKeyBits) | ((uint32_t)k << 30);
  uint32_t h = __umulhi(key * 0x9E3779B1u, m);
#if GALE_CHECK_BOUNDS
  uint32_t probe = 0;
#endif
  for (;;) {  // a table has at least as many slots as records: an empty slot or the key is always met
    const uint32_t old = atomicCAS(tbl + h, kEmpty32, word);
    if (old == kEmpty32) return;
    if ((old & FB::kKeyMask) == key) {
      const int s2 = (int)((old >> FB::kKeyBits) & FB::kIdxMask), k2 = (int)(old >> 30);
      if (!GALE_IN_BOUNDS(err, s2 < s_all && k2 < D)) return;
      // an external simplex only ever records its facet 0
      const int i1 = s < R.s_ext ? s : R.xpad + (s - R.s_ext) * D + k;
      const int i2 = s2 < R.s_ext ? s2 : R.xpad + (s2 - R.s_ext) * D + k2;
      const int g1 = s < R.s_ext ? R.texid[s] : R.t_lo + (s - R.s_ext);
      const int g2 = s2 < R.s_ext ? R.texid[s2] : R.t_lo + (s2 - R.s_ext);
      if (!GALE_IN_BOUNDS(err, i1 >= 0 && i1 < R.cap && i2 >= 0 && i2 < R.cap)) return;
      R.res[i1] = g2;
      R.res[i2] = g1;
      return;
    }
    h = h + 1 == m ? 0u : h + 1;
#if GALE_CHECK_BOUNDS
    if (++probe >= m) { raise_err(err, ERR_TT_TABLE_FULL); return; }
#endif
  }
}

// Key of the facet opposite local vertex K: the facet's vertices other than its lowest one.
template <int D, int K>
__device__ __forceinline__ uint32_t facet_key(const int (&l)[4]) {
  if constexpr (D == 4) {
    const int a = K <= 1 ? l[2] : l[1];
    const int b = K == 3 ? l[2] : l[3];
    return (uint32_t)a | ((uint32_t)b << 9);
  } else {
    return (uint32_t)(K <= 1 ? l[2] : l[1]);
  }
}

// Staging area -> global with one TMA bulk store for the 16-byte aligned body and scalar stores for
// the ragged ends. Staging element j corresponds to global element (g0 - mis) + j, j in [mis, mis+n),
// mis = g0 & 3, so the two addresses share their 16-byte phase. One thread calls this.
__device__ __forceinline__ void bulk_emit(int32_t* gbase, long long g0, int n, const int32_t* stage, int mis) {
  const int jb = (mis + 3) & ~3, je = (mis + n) & ~3;
  int32_t* g = gbase + (g0 - mis);
  if (je > jb) bulk_s2g(g + jb, stage + jb, (uint32_t)(je - jb) * 4u);
  bulk_commit();
  const int head_end = min(jb, mis + n);
  for (int j = mis; j < head_end; ++j) GALE_ST(g + j, stage[j]);
  for (int j = max(je, jb); j < mis + n; ++j) GALE_ST(g + j, stage[j]);
}

// ------------------------------------------------------------------------------------------------
// The batch kernel: VT + VV + TT for every tile of the requested clusters (or, COUNT, the exact
// VT / VV sizes of tiles [tile_base, tile_base + gridDim.x) — the paper's leader producer likewise
// sizes its relation arrays before launch). NT >= rows per tile.
template <int D, int NT, bool COUNT, int LB>
__global__ void __launch_bounds__(NT, (NT <= 128 ? 8 : 4))
gale_batch_kernel(const DeviceMesh M, const __grid_constant__ BatchParams P, const SmemCfg C,
                  const SmemLayout L, const OutPtrs O) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t mask = P.mask;
  const bool do_vt = !COUNT && (mask & REL_VT) != 0, do_vv = (mask & REL_VV) != 0;
  const bool do_tt = !COUNT && (mask & REL_TT) != 0;

  // ---- block -> (cluster slot, tile): worked out by the first warp, shared through BlockCtx ------
  if (!COUNT) {
    if (blockIdx.x == 0 && tid == 0) {  // terminal offsets (also covers batches without rows)
      if (do_vt) { O.vt_offsets[0] = 0; O.vt_offsets[P.total_rows] = P.total_vt_nnz; }
      if (do_vv) { O.vv_offsets[0] = 0; O.vv_offsets[P.total_rows] = P.total_vv_nnz; }
    }
    if ((int)blockIdx.x >= P.tile_prefix[P.n_clusters]) return;
  }
  BlockCtx* ctx = reinterpret_cast<BlockCtx*>(smem + L.ctx);
  void* bar = smem + L.mbar;
  if (tid < 32) {
    int slot = 0, tile;
    if (COUNT) {
      tile = P.tile_base + (int)blockIdx.x;
    } else {
      if (P.uniform_tiles > 0) {
        slot = (int)blockIdx.x / P.uniform_tiles;
      } else {
        int lo = 0, hi = P.n_clusters;
        while (hi - lo > 1) {
          const int mid = (lo + hi) >> 1;
          if (P.tile_prefix[mid] <= (int)blockIdx.x) lo = mid; else hi = mid;
        }
        slot = lo;
      }
      tile = __ldg(M.cluster_tile_begin + P.cluster[slot]) + ((int)blockIdx.x - P.tile_prefix[slot]);
    }
    if (lane < (int)(sizeof(TileDesc) / 16))
      reinterpret_cast<int4*>(&ctx->td)[lane] = __ldg(reinterpret_cast<const int4*>(M.tiles + tile) + lane);
    __syncwarp();
    if (lane == 0) {
      const TileDesc& t = ctx->td;
      ctx->tile = tile;
      if (!COUNT) {
        ctx->row0 = P.row_base[slot] + t.row_rel;
        ctx->vt0 = P.vt_base[slot] + t.vt_rel;
        ctx->vv0 = P.vv_base[slot] + t.vv_rel;
        ctx->tt0 = P.tt_base[slot] + t.tt_rel;
        ctx->tt_slot = P.tt_base[slot];
      }
      // P0a: stage the tile's lists with TMA bulk copies; completion is counted on the mbarrier
      const int S0 = t.s_int + t.s_ext;
      mbar_init(bar, 1);
      fence_proxy_async();
      const uint32_t b_t = (uint32_t)((S0 + 3) & ~3) * (4u * LB);
      const uint32_t b_x = COUNT ? 0u : (uint32_t)((t.s_ext + 3) & ~3) * 4u;
      const uint32_t b_g = (!COUNT && (do_vv || do_tt || C.stage_t)) ? (uint32_t)((t.nloc + 3) & ~3) * 4u : 0u;
      mbar_arrive_expect_tx(bar, (C.stage_t ? 0u : b_t) + b_x + b_g);
      if (b_t && !C.stage_t) bulk_g2s(smem + L.tets, static_cast<const unsigned char*>(M.loc) + t.stg_off * (4 * LB), b_t, bar);
      if (b_x) bulk_g2s(smem + L.texid, M.tex + t.tex_off, b_x, bar);
      if (b_g) bulk_g2s(smem + L.gid, M.gid + t.gid_off, b_g, bar);
    }
  }
  // P0b: clear (needs nothing of the tile's record)
  {
    int4* z = reinterpret_cast<int4*>(smem + L.bmT);
    const int n16 = (L.zero_end - L.bmT) >> 4;
    for (int i = tid; i < n16; i += NT) z[i] = make_int4(0, 0, 0, 0);
  }
  if (do_tt) {  // tables empty, TT rows "none": both all-ones, contiguous
    int4* z = reinterpret_cast<int4*>(smem + L.tbl);
    const int n16 = (L.ones_end - L.tbl) >> 4;
    for (int i = tid; i < n16; i += NT) z[i] = make_int4(-1, -1, -1, -1);
  }
  if (tid == 0) { reinterpret_cast<uint32_t*>(smem + L.misc)[0] = 0u; reinterpret_cast<uint32_t*>(smem + L.misc)[1] = 0u; }
  __syncthreads();
  const TileDesc& td = ctx->td;
  const int tile = ctx->tile;
  const int nrows = td.nrows, t_lo = td.t_lo, s_int = td.s_int, s_ext = td.s_ext, nlo = td.nlo;
  const int S = s_int + s_ext;
  const int WT = C.WT, WV = C.WV;
  const int wT = (S + 31) >> 5, wV = (td.nloc + 31) >> 5;
#if GALE_CHECK_BOUNDS
  {
    bool ok = nrows >= 0 && nrows <= C.tv && NT >= C.tv && S >= 0 && S <= C.smax && nlo >= 0 &&
              nlo + nrows <= td.nloc && wT <= WT;
    if (!COUNT) ok = ok && s_ext <= C.sext && td.nloc <= C.nloc;  // count mode stages neither T_ex ids nor the vertex table
    if (mask & REL_VV) ok = ok && wV <= WV;
    if (do_tt) ok = ok && s_int <= C.sint && ((s_ext + 3) & ~3) <= C.sext && td.vt_nnz + (D - 2) * s_int <= C.tbl;
    if (do_vt) ok = ok && td.vt_nnz <= C.vt_max;
    if (!COUNT && (mask & REL_VV)) ok = ok && td.vv_nnz <= C.vv_max;
    if (!ok) {  // block-uniform: leave before anything is staged
      if (tid == 0) raise_err(M.err, ERR_BOUNDS);
      return;
    }
  }
#endif

  unsigned char* tets = smem + L.tets;
  int32_t* texid = reinterpret_cast<int32_t*>(smem + L.texid);
  int32_t* gid = reinterpret_cast<int32_t*>(smem + L.gid);
  int32_t* ft = reinterpret_cast<int32_t*>(smem + L.ft);          // first_tet[v_lo .. v_lo+nrows]
  int32_t* offT = reinterpret_cast<int32_t*>(smem + L.offT);      // VT offsets of the tile's rows (+ total)
  int32_t* offV = reinterpret_cast<int32_t*>(smem + L.offV);
  int32_t* runpos = reinterpret_cast<int32_t*>(smem + L.runpos);  // VT position of simplex t of row r's run = runpos[r] + t
  int32_t* tbo = reinterpret_cast<int32_t*>(smem + L.tbo);        // facet-table offsets of the rows (+ total)
  uint32_t* scan = reinterpret_cast<uint32_t*>(smem + L.scan);
  uint32_t* misc = reinterpret_cast<uint32_t*>(smem + L.misc);    // [0] chunk counter, [1] fallback queue length
  uint32_t* bmT = reinterpret_cast<uint32_t*>(smem + L.bmT);
  uint32_t* bmV = reinterpret_cast<uint32_t*>(smem + L.bmV);
  uint16_t* pfx = reinterpret_cast<uint16_t*>(smem + L.pfx);      // set bits of the row before word w
  uint32_t* tbl = reinterpret_cast<uint32_t*>(smem + L.tbl);
  unsigned char* dflag = smem + L.dflag;  // external simplex s: this tile writes its TT entry 0 (see P4)
  TTRes R;                                // TT results as global ids, -1 = none
  R.res = reinterpret_cast<int32_t*>(smem + L.ttres);
  R.texid = texid; R.s_ext = s_ext; R.xpad = (s_ext + 3) & ~3; R.t_lo = t_lo;
  R.cap = C.sext + C.sint * D;
  int32_t* st_vt = reinterpret_cast<int32_t*>(smem + L.st_vt);
  int32_t* st_vv = reinterpret_cast<int32_t*>(smem + L.st_vv);
  uint16_t* fbq = reinterpret_cast<uint16_t*>(smem + L.fbq);

  const int row0 = ctx->row0, vt0 = ctx->vt0, vv0 = ctx->vv0, tt0 = ctx->tt0;
  const int mis_vt = vt0 & 3, mis_vv = vv0 & 3;  // 16-byte phase of the tile's output segments
  for (int i = tid; i <= nrows; i += NT) ft[i] = __ldg(M.first_tet + td.v_lo + i);  // read in P2, after a barrier
  mbar_wait(bar, 0);
  if (!COUNT && C.stage_t) {
    // A/B of the create-time re-encoding (SURVEY §8 a1 as written): read the rows of T themselves —
    // internal ones are contiguous, external ones are gathered through T_ex — and map every vertex to
    // its tile-local id here: tile vertices by subtraction, halo vertices by binary search in the
    // staged vertex table (sorted: [halo below][tile][halo above]).
    const int up0 = nlo + nrows, nloc = td.nloc;
    for (int s = tid; s < S; s += NT) {
      const long long t = s < s_ext ? texid[s] : t_lo + (s - s_ext);
      uint32_t l[4] = {LB == 1 ? 0xFFu : 0xFFFFu, LB == 1 ? 0xFFu : 0xFFFFu, LB == 1 ? 0xFFu : 0xFFFFu, LB == 1 ? 0xFFu : 0xFFFFu};
      int v[D];
      if constexpr (D == 4) {
        const int4 q = __ldg(reinterpret_cast<const int4*>(M.T) + t);
        v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
      } else {
#pragma unroll
        for (int k = 0; k < D; ++k) v[k] = __ldg(M.T + t * D + k);
      }
#pragma unroll
      for (int k = 0; k < D; ++k) {
        const int r = v[k] - td.v_lo;
        if ((unsigned)r < (unsigned)nrows) { l[k] = (uint32_t)(nlo + r); continue; }
        int lo = r < 0 ? 0 : up0, hi = r < 0 ? nlo : nloc;
        while (lo < hi) {
          const int mid = (lo + hi) >> 1;
          if (gid[mid] < v[k]) lo = mid + 1; else hi = mid;
        }
        l[k] = (uint32_t)lo;
      }
      if constexpr (LB == 1) reinterpret_cast<uint32_t*>(tets)[s] = l[0] | (l[1] << 8) | (l[2] << 16) | (l[3] << 24);
      else reinterpret_cast<uint2*>(tets)[s] = make_uint2(l[0] | (l[1] << 16), l[2] | (l[3] << 16));
    }
    __syncthreads();
  }

  // ---- P1: VT incidence bits and VV bits, one thread per staged simplex ------------------------
  const uint32_t aT = smem_u32(bmT), aV = smem_u32(bmV);
  const uint32_t strideT = (uint32_t)WT * 4u, strideV = (uint32_t)WV * 4u;
  // Consecutive staged simplices share most of their vertices at the same positions, so neighbouring
  // lanes would OR into the same bitmap row in the same instruction (shared-memory atomics on one word
  // serialise: measured 3.1 of 4.0 wavefronts per tet were such conflicts). Each lane therefore visits
  // its vertices in an order rotated by its lane number (one PRMT on the packed 8-bit ids); the marking
  // is symmetric in the position, only "k is not the lowest vertex" has to follow the rotation (k0).
  int rot = 0, k0 = 0;
  uint32_t rot_sel = 0x3210u;
  if constexpr (LB == 1) {
    rot = D == 4 ? (lane & 3) : (lane % 3);
    k0 = rot == 0 ? 0 : D - rot;  // where the lowest vertex ends up
    rot_sel = D == 4 ? ((0x32103210u >> (rot * 4)) & 0xFFFFu) : (rot == 0 ? 0x3210u : (rot == 1 ? 0x3021u : 0x3102u));
  }
  for (int s = tid; s < S; s += NT) {
    int l[4];
    if constexpr (LB == 1) {
      const uint32_t q = __byte_perm(reinterpret_cast<const uint32_t*>(tets)[s], 0u, rot_sel);
      l[0] = q & 0xFF; l[1] = (q >> 8) & 0xFF; l[2] = (q >> 16) & 0xFF; l[3] = q >> 24;
    } else {
      load_local<LB>(tets, s, l);
    }
#if GALE_CHECK_BOUNDS
    for (int k = 0; k < D; ++k)
      if (!GALE_IN_BOUNDS(M.err, l[k] >= 0 && l[k] < td.nloc)) l[k] = nlo;  // keep later indexing inside the row
    if (s >= s_ext) (void)GALE_IN_BOUNDS(M.err, (unsigned)(l[k0] - nlo) < (unsigned)nrows);  // internal: lowest vertex in the tile
#endif
    const uint32_t col = aT + (uint32_t)(s >> 5) * 4u;
    const uint32_t bit = 1u << (s & 31);
    int r[D];
#pragma unroll
    for (int k = 0; k < D; ++k) r[k] = l[k] - nlo;
#pragma unroll
    for (int k = 0; k < D; ++k)
      red_or_shared_if(k != k0 && (unsigned)r[k] < (unsigned)nrows, col + (uint32_t)r[k] * strideT, bit);
    if (do_vv) {
      uint32_t w[D], b[D];
#pragma unroll
      for (int j = 0; j < D; ++j) { w[j] = ((uint32_t)l[j] >> 5) * 4u; b[j] = 1u << (l[j] & 31); }
#pragma unroll
      for (int k = 0; k < D; ++k) {
        const bool in = (unsigned)r[k] < (unsigned)nrows;
        const uint32_t row = aV + (uint32_t)r[k] * strideV;
#pragma unroll
        for (int j = 0; j < D; ++j)
          if (j != k) red_or_shared_if(in, row + w[j], b[j]);  // "each other vertex"
      }
    }
  }
  __syncthreads();

  // ---- P2: per row prefix counts and degrees -> offsets ----------------------------------------
  int n_vt, n_vv;
  int my_offV = 0;
  {
    uint32_t deg = 0u, degv = 0u;
    int nb = 0;
    if (tid < nrows) {
      const uint32_t* row = bmT + tid * WT;
      uint16_t* pf = pfx + tid * WT;
      for (int w = 0; w < wT; ++w) {
        pf[w] = (uint16_t)nb;
        nb += __popc(row[w]);
      }
      deg = (uint32_t)(nb + ft[tid + 1] - ft[tid]);
      if (do_vv) {
        const uint32_t* rv = bmV + tid * WV;
        for (int w = 0; w < wV; ++w) degv += __popc(rv[w]);
      }
    }
    uint32_t tot = 0u, ex = 0u;
    if (C.tv <= 32) {  // the rows fit one warp: no block-wide scan, no barriers
      if (tid < 32) {
        const uint32_t x = deg | (degv << 16);
        uint32_t inc = x;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, inc, d);
          if (lane >= d) inc += y;
        }
        tot = __shfl_sync(0xFFFFFFFFu, inc, 31);
        ex = inc - x;
      }
    } else {
      ex = block_exclusive_scan<NT>(deg | (degv << 16), scan, &tot);
    }
    n_vt = (int)(tot & 0xFFFFu);
    n_vv = (int)(tot >> 16);
    if (tid < nrows) {
      const int ot = (int)(ex & 0xFFFFu);
      my_offV = (int)(ex >> 16);
      offT[tid] = ot;
      offV[tid] = my_offV;
      runpos[tid] = ot + nb - ft[tid];
      tbo[tid] = ot + (D - 2) * (ft[tid] - t_lo);
      if (do_vt) O.vt_offsets[row0 + tid] = vt0 + ot;
      if (!COUNT && do_vv) O.vv_offsets[row0 + tid] = vv0 + my_offV;
    }
    if (tid == 0) { offT[nrows] = n_vt; offV[nrows] = n_vv; tbo[nrows] = n_vt + (D - 2) * s_int; }
  }
  if (COUNT) {
    if (tid == 0) {
      O.stats[(long long)tile * 4 + 0] = n_vt;
      O.stats[(long long)tile * 4 + 1] = n_vv;
      O.stats[(long long)tile * 4 + 2] = 0;
      O.stats[(long long)tile * 4 + 3] = 0;
    }
    return;
  }
  if (tid == 0 && (((mask & REL_VT) && n_vt != td.vt_nnz) || (do_vv && n_vv != td.vv_nnz)))
    raise_err(M.err, ERR_SIZE_MISMATCH);  // the sizes fixed at create must be reproduced exactly
  __syncthreads();
  n_vt = offT[nrows];  // (the scan's totals are only known to the scanning threads)
  n_vv = offV[nrows];

  const int c_lo = td.v_lo - td.row_rel, c_hi = c_lo + td.c_rows;  // the cluster's vertex range
  const int c_tlo = t_lo - td.tt_rel;                               // its first internal simplex
  const int tile_hi = nlo + nrows;
  // ---- P3a: TT facet records into the per-vertex tables -----------------------------------------
  if (do_tt) {
    // facet 0 of every staged simplex whose second vertex is a tile vertex
    for (int s = tid; s < S; s += NT) {
      int l[4];
      load_local<LB>(tets, s, l);
#if GALE_CHECK_BOUNDS
      for (int k = 0; k < D; ++k)
        if (l[k] < 0 || l[k] >= td.nloc) l[k] = nlo;  // reported in P1
#endif
      const int r1 = l[1] - nlo;
      if ((unsigned)r1 < (unsigned)nrows) {  // facet 0 has lowest vertex l[1]
        const int b0 = tbo[r1];
        const uint32_t m = (uint32_t)(tbo[r1 + 1] - b0);
        // an external simplex of this cluster: its own tile cannot see this facet, so this tile writes
        // entry 0 of its TT row (P4)
        if (s < s_ext && gid[l[0]] >= c_lo) dflag[s] = 1;
        if (GALE_IN_BOUNDS(M.err, b0 >= 0 && b0 + (int)m <= C.tbl))
          facet_place<D>(tbl + b0, m, facet_key<D, 0>(l), s, 0, R, S, M.err);
      }
    }
    // facets 1..D-1 of the internal simplices: their lowest vertex is l[0], a tile vertex. One thread per
    // record, every lane busy.
    const int nrec = (D - 1) * s_int;
    for (int i = tid; i < nrec; i += NT) {
      const int q = i / (D - 1);
      const int k = 1 + (i - q * (D - 1));
      const int s = s_ext + q;
      int l[4];
      load_local<LB>(tets, s, l);
#if GALE_CHECK_BOUNDS
      for (int kk = 0; kk < D; ++kk)
        if (l[kk] < 0 || l[kk] >= td.nloc) l[kk] = nlo;
#endif
      const int r = l[0] - nlo;
      if (!GALE_IN_BOUNDS(M.err, (unsigned)r < (unsigned)nrows)) continue;
      uint32_t key;
      if constexpr (D == 4) key = (uint32_t)(k == 1 ? l[2] : l[1]) | ((uint32_t)(k == 3 ? l[2] : l[3]) << 9);
      else key = (uint32_t)(k == 1 ? l[2] : l[1]);
      const int b0 = tbo[r];
      const uint32_t m = (uint32_t)(tbo[r + 1] - b0);
      if (GALE_IN_BOUNDS(M.err, b0 >= 0 && b0 + (int)m <= C.tbl)) facet_place<D>(tbl + b0, m, key, s, k, R, S, M.err);
    }
    __syncthreads();  // the tables are dead from here on: the VT / VV staging areas reuse their bytes
  }

  // ---- P3b: VV rows -> staging; per staged simplex: VT scatter by rank ----------------------------
  if (do_vv && tid < nrows) {
    const uint32_t* row = bmV + tid * WV;
    int pos = mis_vv + my_offV;
    for (int w = 0; w < wV; ++w) {
      uint32_t bits = row[w];
      while (bits) {
        const int lid = (w << 5) + __ffs(bits) - 1;
        bits &= bits - 1;
        if (GALE_IN_BOUNDS(M.err, pos < C.vv_max + 4 && lid < td.nloc)) st_vv[pos] = gid[lid];
        ++pos;
      }
    }
  }
  if (do_vt) {
    // 32-simplex chunks go to the warps round-robin; the warps that expanded VV rows above sit out the
    // first round (an expansion is about one chunk's work)
    const int nexp = do_vv ? (nrows + 31) >> 5 : 0;
    const uint32_t aSt = smem_u32(st_vt + mis_vt);
    const int warp = tid >> 5;
    for (int j = warp < nexp ? warp + NT / 32 : warp;; j += NT / 32) {
      const int base = (j - nexp) << 5;
      if (base >= S) break;
      const int s = base + lane;
      if (s >= S) continue;
      int l[4];
      load_local<LB>(tets, s, l);
#if GALE_CHECK_BOUNDS
      for (int k = 0; k < D; ++k)
        if (l[k] < 0 || l[k] >= td.nloc) l[k] = nlo;  // reported in P1
#endif
      const bool internal = s >= s_ext;
      const int g = internal ? t_lo + (s - s_ext) : texid[s];
      const int w = s >> 5;
      const uint32_t below = (1u << (s & 31)) - 1u;
#pragma unroll
      for (int k = 1; k < D; ++k) {  // branch-free: lanes outside the tile read row 0 and skip the store
        const int r = l[k] - nlo;
        const bool in = (unsigned)r < (unsigned)nrows;
        const int rr = in ? r : 0;
        const int pos = offT[rr] + (int)pfx[rr * WT + w] + __popc(bmT[rr * WT + w] & below);
        st_shared_if(in && GALE_IN_BOUNDS(M.err, pos >= 0 && pos < C.vt_max), aSt + (uint32_t)pos * 4u, g);
      }
      {
        const int rr = internal ? l[0] - nlo : 0;
        const int pos = runpos[rr] + g;
        st_shared_if(internal && GALE_IN_BOUNDS(M.err, (unsigned)rr < (unsigned)nrows && pos >= 0 && pos < C.vt_max),
                     aSt + (uint32_t)pos * 4u, g);
      }
    }
  }
  fence_proxy_async();  // staging areas were written through the generic proxy, TMA reads them
  __syncthreads();

  // ---- P4: write-out ---------------------------------------------------------------------------
  if (do_vt && tid == 0) bulk_emit(O.vt_indices, vt0, n_vt, st_vt, mis_vt);
  if (do_vv && tid == 32) bulk_emit(O.vv_indices, vv0, n_vv, st_vv, mis_vv);

  if (do_tt) {
    // TT rows of the internal simplices. Entry 0 = -1 means boundary, or a facet (l[1], ..) without a
    // vertex in this tile (l[1] lies above it): only then the simplex is looked at again.
    for (int i = tid; i < s_int; i += NT) {
      int r[D];
      if constexpr (D == 4) {
        const int4 v = reinterpret_cast<const int4*>(R.res + R.xpad)[i];
        r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w;
      } else {
#pragma unroll
        for (int k = 0; k < D; ++k) r[k] = R.res[R.xpad + i * D + k];
      }
      bool out0 = false, delegated = false;
      if (r[0] < 0) {
        int l[4];
        load_local<LB>(tets, s_ext + i, l);
        out0 = l[1] >= tile_hi;
        delegated = out0 && gid[min(l[1], td.nloc - 1)] < c_hi;  // the tile that owns l[1] writes entry 0
      }
      int32_t* o = O.tt_indices + (long long)(tt0 + i) * D;
      if constexpr (D == 4) {
        if (!delegated) {
          GALE_ST(reinterpret_cast<int4*>(o), make_int4(r[0], r[1], r[2], r[3]));
        } else {
          GALE_ST(o + 1, r[1]);
          GALE_ST(reinterpret_cast<int2*>(o + 2), make_int2(r[2], r[3]));
        }
      } else {
        if (!delegated) GALE_ST(o, r[0]);
        GALE_ST(o + 1, r[1]);
        GALE_ST(o + 2, r[2]);
      }
      if (out0 && !delegated) {  // cross-cluster facet: resolved from global memory below
        const uint32_t q = atomicAdd(&misc[1], 1u);
        if (GALE_IN_BOUNDS(M.err, (int)q < C.sint)) fbq[q] = (uint16_t)i;
      }
    }
    // entry 0 of the flagged external simplices (same cluster, second vertex in this tile)
    for (int s = tid; s < s_ext; s += NT)
      if (dflag[s]) {
        const long long row = (long long)ctx->tt_slot + (texid[s] - c_tlo);
        GALE_ST(O.tt_indices + row * D, R.res[s]);
      }
    __syncthreads();  // queue complete, TT rows stored
    // ---- a5: one queued facet per thread, resolved from global memory -------------------------
    const int nq = (int)misc[1];
    for (int q = tid; q < nq; q += NT) {
      const int i = fbq[q];
      int l[4];
      load_local<LB>(tets, s_ext + i, l);
      const int t = t_lo + i;
      const int b = gid[l[1]], c = gid[l[2]], d = D == 4 ? gid[l[3]] : 0;
      const int f0 = __ldg(M.first_tet + b), f1 = __ldg(M.first_tet + b + 1);
      const int r = tt_fallback<D>(M, f0, f1, b, c, d, t);
      if (r >= 0) O.tt_indices[(long long)(tt0 + i) * D] = r;  // ordered after the row store by the barrier
    }
  }
  // the block's shared memory must stay intact until the bulk stores have read it
  if (tid == 0 || tid == 32) bulk_wait_read_all();
}

}  // namespace gale
