// gale_walk.cuh — the "walk" variant of the batch kernel (same inputs, same outputs as gale_batch_kernel).
//
// Two threads per tile vertex p walk p's incidences serially: thread A(p) the set bits of p's VT bitmap
// row (= VT(p) without its run, already sorted), thread B(p) the run of p. The thread owns its row, so
// VV bits and TT facet tables need no claiming. This is cheapest when all vertex stars look alike
// (regular grids: every lane of a warp has the same amount of work); on irregular meshes the lanes of a
// warp wait for the heaviest vertex and the per-vertex capacities are dictated by it — there the dense
// kernel (gale_kernels.cuh, one thread per staged simplex) wins. gale_mesh_create times both on a sample
// batch and keeps the faster one.
//
// Phases: P0 one warp works out the tile and stages its lists with TMA bulk copies, the others clear; P1 VT incidence bits, one thread per staged simplex;
// P2 row degrees -> scan -> VT offsets; P3 A(p): walk the bits: VT entries + VV bits + flag "p is the
// second vertex"; B(p): walk the run: VT entries, VV bits, facet records 1..D-1 into p's private table;
// P4 A(p): facets 0 of the flagged simplices join p's table (both cofaces of a facet with lowest vertex
// p have p as lowest or second-lowest vertex, so the second arrival meets the first); B(p): VV row ->
// degree -> scan -> expansion; P5 translate to global ids, coalesced write-out; facets (l[1], ..) with
// l[1] outside the tile: same cluster -> written by the tile that owns l[1] (it has the simplex in its
// T_ex list; the entry goes to the output when the facet is placed or matched), else resolved from global
// memory (a5).
// Shared-memory layout: what a thread owns alone — its rows of the VT and VV bitmaps, the facet table of its
// vertex — is stored word-interleaved over the rows (word w of row p at [w * TV + p]): lane p always works in
// bank p. Config 5: 11.2 KB per block, 48 registers, 19 resident blocks of 64 threads per SM.
#pragma once
#include "gale_kernels.cuh"

namespace gale {

struct WalkLayout {
  int mbar, ctx, tets, texid, gid, fbq, scan, bmT, bmV, bm_end;
  int tbl, ttrow, tt_end;
  int st_vt, st_vv;
  int total;
};

// Rows per block of the instantiation that runs tiles of `tv` vertices (NT / 2, a multiple of 32).
__host__ __device__ inline int walk_rows_for_tile(int tv) { return tv > 128 ? 256 : (tv > 64 ? 128 : (tv > 32 ? 64 : 32)); }

// Capacities come in a SmemCfg; `hs` = table slots per tile vertex. The structures a thread owns alone (VV
// bitmap row, facet table of vertex p) are stored word-interleaved over the rows — word w of row p at
// [w * TV + p] — so that lane p always works in bank p and the serial walks meet no bank conflict.
template <int D>
__host__ __device__ inline WalkLayout make_walk_layout(const SmemCfg& c) {
  WalkLayout L;
  const int tvp = walk_rows_for_tile(c.tv);
  int o = 0;
  L.mbar = o;   o = align16(o + 8);
  L.ctx = o;    o = align16(o + 112);
  L.tets = o;   o = align16(o + c.smax * 4 * c.lb);
  L.texid = o;  o = align16(o + c.sext * 4);
  L.gid = o;    o = align16(o + c.nloc * 4);  // (the slice of I_T is read straight from global memory)
  L.scan = o;   o = align16(o + 36 * 4);   // [0..33) scan scratch, [33] a5 queue length, [34] n_vv; every thread counts its own row
  // VT bitmap (P1-P3); afterwards the same bytes hold the VV staging area (written in P4) and the
  // fallback queue (written in P5)
  L.bmT = o;
  {
    const int bm = align16(tvp * ((c.smax + 31) / 32) * 4);  // word w of row p at [w * TV + p], like the VV rows
    L.st_vv = o;
    L.fbq = o + align16(c.vv_max * 2);
    const int reuse = align16(c.vv_max * 2) + align16(c.sint * 2);
    o += bm > reuse ? bm : reuse;
  }
  L.bmV = o;    o = align16(o + (c.WV ? tvp * ((c.nloc + 31) / 32) * 4 : 0));  // interleaved rows need no odd stride
  L.bm_end = o;
  L.tbl = o;    o = align16(o + (c.hs ? tvp * c.hs * 4 : 0));
  L.ttrow = o;  o = align16(o + (c.hs ? c.sint * D * 2 : 0));
  L.tt_end = o;
  L.st_vt = o;  o = align16(o + c.vt_max * 2);
  L.total = o;
  return L;
}

// Barrier among the `count` threads that name the same id (ids 1..15; 0 is __syncthreads).
__device__ __forceinline__ void named_barrier(int id, int count) {
  asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(count) : "memory");
}

__device__ __forceinline__ uint32_t bit_of(int l) { return 1u << (l & 31); }

struct GroupCtx {
  uint32_t* tbl;       // this vertex's table, hs slots, slot h at tbl[h * TV]
  uint32_t hs;         // slots (any size >= the group's records: a group never overflows its table)
  uint16_t* ttrow;     // TT rows of the tile's internal simplices as staged indices, 0xFFFF = none
  int s_ext;
  int s_all;           // staged simplices of the tile (bounds-checked build)
  // entry 0 of an external simplex of this cluster goes straight to the output (its row belongs to another tile)
  const unsigned char* tets;
  const int32_t* texid;
  const int32_t* gid;
  int32_t* tt;         // O.tt_indices
  int t_lo, tt_slot, c_lo, c_tlo;
};

// TT entry 0 of the external simplex s (its facet 0 has this tile's vertex p as lowest vertex, so only this tile
// can match it): written when s belongs to this tile's cluster (else the cluster of s resolves it itself, a5).
// partner = staged index of the coface, -1 = none so far: the first arrival of a facet writes -1 and the same
// thread overwrites it if the coface turns up later (same thread, same address: program order).
template <int D, int LB>
__device__ __forceinline__ void ext_entry0(const GroupCtx& g, int s, int partner) {
  const int l0 = LB == 2 ? (int)reinterpret_cast<const uint16_t*>(g.tets)[s * 4] : (int)g.tets[s * 4];
  if (g.gid[l0] >= g.c_lo) {
    const int val = partner < 0 ? -1 : (partner < g.s_ext ? g.texid[partner] : g.t_lo + (partner - g.s_ext));
    GALE_ST(g.tt + (long long)(g.tt_slot + (g.texid[s] - g.c_tlo)) * D, val);
  }
}

// Place facet k of staged simplex s with key `key`: claim an empty slot, or meet the record that
// holds the same key (the other coface) and write both TT entries. The thread owns the table.
template <int D, int TV, int LB>
__device__ __forceinline__ void group_place(const GroupCtx& g, uint32_t key, int s, int k, int32_t* err) {
  using FB = FacetBits<D>;
  uint32_t h = __umulhi(key * 0x9E3779B1u, g.hs);
  uint32_t cur = g.tbl[h * TV];
#if GALE_CHECK_BOUNDS
  uint32_t probe = 0;
#endif
  // a table has more slots than its group has records, so an empty slot or the key is always met
  while (cur != kEmpty32 && (cur & FB::kKeyMask) != key) {  // probe loop kept minimal: lanes diverge here
    h = h + 1 == g.hs ? 0u : h + 1;
    cur = g.tbl[h * TV];
#if GALE_CHECK_BOUNDS
    if (++probe >= g.hs) { raise_err(err, ERR_TT_TABLE_FULL); return; }
#endif
  }
  if (!GALE_IN_BOUNDS(err, h < g.hs && (uint32_t)s <= FB::kIdxMask && key <= FB::kKeyMask && k >= 0 && k < D)) return;
  if (cur == kEmpty32) {
    g.tbl[h * TV] = key | ((uint32_t)s << FB::kKeyBits) | ((uint32_t)k << 30);
    if (s < g.s_ext) ext_entry0<D, LB>(g, s, -1);
  } else {
    const int s2 = (int)((cur >> FB::kKeyBits) & FB::kIdxMask), k2 = (int)(cur >> 30);
    if (!GALE_IN_BOUNDS(err, s < g.s_all && s2 < g.s_all && k2 < D)) return;
    // an external simplex only ever records its facet 0
    if (s >= g.s_ext) g.ttrow[(s - g.s_ext) * D + k] = (uint16_t)s2; else ext_entry0<D, LB>(g, s, s2);
    if (s2 >= g.s_ext) g.ttrow[(s2 - g.s_ext) * D + k2] = (uint16_t)s; else ext_entry0<D, LB>(g, s2, s);
  }
}

// Exclusive scan over the B half of the block (threads [NT/2, NT)), one value per thread, with a
// named barrier so that the A half is not held up. Returns the exclusive prefix; *total = sum.
template <int NT>
__device__ __forceinline__ uint32_t half_exclusive_scan(uint32_t x, uint32_t* scratch, uint32_t* total) {
  constexpr int TV = NT / 2;
  const int lane = threadIdx.x & 31, warp = (threadIdx.x - TV) >> 5;
  uint32_t inc = x;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, inc, d);
    if (lane >= d) inc += y;
  }
  if constexpr (TV <= 32) {
    *total = __shfl_sync(0xFFFFFFFFu, inc, 31);
    return inc - x;
  } else {
    constexpr int NW = TV / 32;
    if (lane == 31) scratch[warp] = inc;
    named_barrier(1, TV);
    uint32_t base = 0u, tot = 0u;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const uint32_t v = scratch[w];
      if (w < warp) base += v;
      tot += v;
    }
    named_barrier(1, TV);  // scratch may be reused
    *total = tot;
    return base + inc - x;
  }
}

// NT = 2 * (rows per tile capacity): thread tid < NT/2 is A(tid), thread NT/2 + p is B(p).
// ALL: the launch computes all three relations (the mask tests fold at compile time).
template <int D, int NT, int LB, bool ALL>
__global__ void __launch_bounds__(NT, (NT <= 64 ? 16 : (NT <= 128 ? 8 : (NT <= 256 ? 4 : 2))))
gale_walk_kernel(const DeviceMesh M, const __grid_constant__ BatchParams P, const SmemCfg C,
                 const WalkLayout L, const OutPtrs O) {
  extern __shared__ __align__(16) unsigned char smem[];
  constexpr int TV = NT / 2;
  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t mask = P.mask;
  const bool do_vt = ALL || (mask & REL_VT) != 0, do_vv = ALL || (mask & REL_VV) != 0, do_tt = ALL || (mask & REL_TT) != 0;
  const bool entries = do_vt || do_tt;  // VT entries are staged (TT reads their flags)

  // ---- block -> (cluster slot, tile): worked out by the first warp, shared through BlockCtx; the same
  // warp issues the TMA bulk copies of the tile's lists (P0a) -------------------------------------
  if (blockIdx.x == 0 && tid == 0) {  // terminal offsets (also covers batches without rows)
    if (do_vt) { O.vt_offsets[0] = 0; O.vt_offsets[P.total_rows] = P.total_vt_nnz; }
    if (do_vv) { O.vv_offsets[0] = 0; O.vv_offsets[P.total_rows] = P.total_vv_nnz; }
  }
  if ((int)blockIdx.x >= P.tile_prefix[P.n_clusters]) return;
  BlockCtx* ctx = reinterpret_cast<BlockCtx*>(smem + L.ctx);
  void* bar = smem + L.mbar;
  if (tid < 32) {
    int slot = 0;
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
    const int tile = __ldg(M.cluster_tile_begin + P.cluster[slot]) + ((int)blockIdx.x - P.tile_prefix[slot]);
    if (lane < (int)(sizeof(TileDesc) / 16))
      reinterpret_cast<int4*>(&ctx->td)[lane] = __ldg(reinterpret_cast<const int4*>(M.tiles + tile) + lane);
    __syncwarp();
    if (lane == 0) {
      const TileDesc& t = ctx->td;
      ctx->tile = tile;
      ctx->row0 = P.row_base[slot] + t.row_rel;
      ctx->vt0 = P.vt_base[slot] + t.vt_rel;
      ctx->vv0 = P.vv_base[slot] + t.vv_rel;
      ctx->tt0 = P.tt_base[slot] + t.tt_rel;
      ctx->tt_slot = P.tt_base[slot];
      mbar_init(bar, 1);
      fence_proxy_async();
      const uint32_t b_t = (uint32_t)((t.s_int + t.s_ext + 3) & ~3) * (4u * LB);
      const uint32_t b_x = (uint32_t)((t.s_ext + 3) & ~3) * 4u;
      const uint32_t b_g = (do_vv || do_tt) ? (uint32_t)((t.nloc + 3) & ~3) * 4u : 0u;
      mbar_arrive_expect_tx(bar, b_t + b_x + b_g);
      if (b_t) bulk_g2s(smem + L.tets, static_cast<const unsigned char*>(M.loc) + t.stg_off * (4 * LB), b_t, bar);
      if (b_x) bulk_g2s(smem + L.texid, M.tex + t.tex_off, b_x, bar);
      if (b_g) bulk_g2s(smem + L.gid, M.gid + t.gid_off, b_g, bar);
    }
  }
  // P0b: clear (needs nothing of the tile's record)
  {
    int4* z = reinterpret_cast<int4*>(smem + L.bmT);
    const int n16 = (L.bm_end - L.bmT) >> 4;
    for (int i = tid; i < n16; i += NT) z[i] = make_int4(0, 0, 0, 0);
  }
  if (do_tt) {  // tables empty, TT rows "none": both all-ones, contiguous
    int4* z = reinterpret_cast<int4*>(smem + L.tbl);
    const int n16 = (L.tt_end - L.tbl) >> 4;
    for (int i = tid; i < n16; i += NT) z[i] = make_int4(-1, -1, -1, -1);
  }
  if (tid == 0) { reinterpret_cast<uint32_t*>(smem + L.scan)[33] = 0u; reinterpret_cast<uint32_t*>(smem + L.scan)[34] = 0u; }
  __syncthreads();
  const TileDesc& td = ctx->td;
  const int nrows = td.nrows, t_lo = td.t_lo, s_int = td.s_int, s_ext = td.s_ext, nlo = td.nlo;
  const int S = s_int + s_ext;
  const int WV = C.WV;
#if GALE_CHECK_BOUNDS
  {
    bool ok = nrows >= 0 && nrows <= C.tv && NT >= 2 * C.tv && S >= 0 && S <= C.smax && s_ext <= C.sext &&
              td.nloc <= C.nloc && nlo >= 0 && nlo + nrows <= td.nloc;
    if (mask & REL_VV) ok = ok && ((td.nloc + 31) >> 5) <= WV;
    if (mask & REL_TT) ok = ok && s_int <= C.sint && C.hs >= 2;
    if (mask & (REL_VT | REL_TT)) ok = ok && td.vt_nnz <= C.vt_max;
    if (mask & REL_VV) ok = ok && td.vv_nnz <= C.vv_max;
    if (!ok) {  // block-uniform: leave before anything is staged
      if (tid == 0) raise_err(M.err, ERR_BOUNDS);
      return;
    }
  }
#endif

  unsigned char* tets = smem + L.tets;
  int32_t* texid = reinterpret_cast<int32_t*>(smem + L.texid);
  int32_t* gid = reinterpret_cast<int32_t*>(smem + L.gid);
  uint16_t* fbq = reinterpret_cast<uint16_t*>(smem + L.fbq);
  uint32_t* scan = reinterpret_cast<uint32_t*>(smem + L.scan);  // [0..33) scans, [33] queue length, [34] n_vv
  uint32_t* bmT = reinterpret_cast<uint32_t*>(smem + L.bmT);
  uint32_t* bmV = reinterpret_cast<uint32_t*>(smem + L.bmV);
  uint32_t* tbl = reinterpret_cast<uint32_t*>(smem + L.tbl);
  uint16_t* ttrow = reinterpret_cast<uint16_t*>(smem + L.ttrow);
  uint16_t* st_vt = reinterpret_cast<uint16_t*>(smem + L.st_vt);
  uint16_t* st_vv = reinterpret_cast<uint16_t*>(smem + L.st_vv);

  const int row0 = ctx->row0, vt0 = ctx->vt0, vv0 = ctx->vv0, tt0 = ctx->tt0;
  mbar_wait(bar, 0);

  // ---- P1: VT incidence bits (rows = tile vertices, columns = staged simplices) ---------------
  // thread t takes the simplices t*K .. t*K+K-1: the lanes of a warp then work K apart in the sorted list, where
  // simplices rarely share a row — neighbouring simplices (same word of the bitmap, same vertices) would hit
  // the same address in one atomic instruction
  const int K1 = (S + NT - 1) / NT;
  for (int s = tid * K1, s_end = min(S, s + K1); s < s_end; ++s) {
    int l[4];
    load_local<LB>(tets, s, l);
#if GALE_CHECK_BOUNDS
    for (int k = 0; k < D; ++k)
      if (!GALE_IN_BOUNDS(M.err, l[k] >= 0 && l[k] < td.nloc)) l[k] = nlo;  // keep later indexing inside the row
    if (s >= s_ext) (void)GALE_IN_BOUNDS(M.err, (unsigned)(l[0] - nlo) < (unsigned)nrows);  // internal: lowest vertex in the tile
#endif
    uint32_t* col = bmT + (s >> 5) * TV;
    const uint32_t bit = bit_of(s);
#pragma unroll
    for (int k = 1; k < D; ++k) {
      const int r = l[k] - nlo;
      if ((unsigned)r < (unsigned)nrows) atomicOr(col + r, bit);
    }
  }
  __syncthreads();

  // ---- P2: row degrees -> VT offsets ----------------------------------------------------------
  const bool isB = tid >= TV;
  const int p = isB ? tid - TV : tid;
  const bool live = p < nrows;
  const int ploc = nlo + p;
  const int wT = (S + 31) >> 5;
  // every thread counts its whole row (conflict-free reads, 12 words on config 5) :
  // no exchange between the halves, no barrier
  int row_bits = 0;
  if (live) {
    const uint32_t* row = bmT + p;
#pragma unroll 4
    for (int w = 0; w < wT; ++w) {
      row_bits += __popc(row[w * TV]);
    }
  }
  int nb = 0, off = 0, n_vt;
  int run_lo = 0, run_hi = 0;  // run of p: simplices [run_lo, run_hi) have p as lowest vertex (I_T)
  {
    uint32_t deg = 0u, tot;
    if (live) {
      nb = row_bits;
      run_lo = __ldg(M.first_tet + td.v_lo + p); run_hi = __ldg(M.first_tet + td.v_lo + p + 1);
      deg = (uint32_t)(nb + run_hi - run_lo);
    }
    if constexpr (NT == 64) {
      // one warp per half, both halves carry the same 32 values: each warp scans for itself, no barrier
      uint32_t inc = deg;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, inc, d);
        if (lane >= d) inc += y;
      }
      n_vt = (int)__shfl_sync(0xFFFFFFFFu, inc, 31);
      off = (int)(inc - deg);
      (void)tot;
    } else {
      const uint32_t ex = block_exclusive_scan<NT>(deg, scan, &tot);  // A and B halves carry the same values
      n_vt = (int)(tot >> 1);
      off = (int)ex - (isB ? n_vt : 0);
    }
  }
  if (do_vt && live && !isB) O.vt_offsets[row0 + p] = vt0 + off;

  // ---- P3: A walks the bits of row p, B walks the run of p ------------------------------------
  uint32_t fmask = 0u;  // A: which of the first 32 entries of the row have p as second vertex (their facets 0 join p's group in P4)
  if (live) {
    uint32_t* vvrow = bmV + p;  // word w of the row at vvrow[w * TV]
    if (!isB) {
      const uint32_t* row = bmT + p;
      int pos = off, sbase = -32;
      uint32_t bits = 0u;
      for (int n = 0; n < nb; ++n) {
        while (bits == 0u) { bits = *row; row += TV; sbase += 32; }
        const int s = sbase + __ffs(bits) - 1;
        bits &= bits - 1;
        int l[4];
        load_local<LB>(tets, s, l);
        const bool second = l[1] == ploc;
        if (n < 32) fmask |= (uint32_t)second << n;
        if (entries && GALE_IN_BOUNDS(M.err, pos >= 0 && pos < C.vt_max && s >= 0 && s < S))
          st_vt[pos++] = (uint16_t)(s | (second ? 0x8000 : 0));
        if (do_vv) {
          // p is not the lowest vertex here: mark l[0] and the D-2 vertices among l[1..D-1] other than p itself
          atomicOr(vvrow + (l[0] >> 5) * TV, bit_of(l[0]));
          const int m1 = second ? l[2] : l[1];
          atomicOr(vvrow + (m1 >> 5) * TV, bit_of(m1));
          if constexpr (D == 4) {
            const int m2 = l[3] == ploc ? l[2] : l[3];
            atomicOr(vvrow + (m2 >> 5) * TV, bit_of(m2));
          }
        }
      }
    } else {
      GroupCtx g;
      if (do_tt) {
        const int hs = C.hs;
        g.tbl = tbl + p;
        g.hs = (uint32_t)hs;
        g.ttrow = ttrow;
        g.tets = tets; g.texid = texid; g.gid = gid; g.tt = O.tt_indices;
        g.t_lo = t_lo; g.tt_slot = ctx->tt_slot; g.c_lo = td.v_lo - td.row_rel; g.c_tlo = t_lo - td.tt_rel;
        g.s_ext = s_ext; g.s_all = S;
      }
      int pos = off + nb;
      const int r1 = run_hi - t_lo;
      for (int i = run_lo - t_lo; i < r1; ++i) {
        const int s = s_ext + i;
        int l[4];
        load_local<LB>(tets, s, l);
        if (entries && GALE_IN_BOUNDS(M.err, pos >= 0 && pos < C.vt_max && s >= s_ext && s < S)) st_vt[pos++] = (uint16_t)s;
        if (do_vv) {
#pragma unroll
          for (int k = 1; k < D; ++k) atomicOr(vvrow + (l[k] >> 5) * TV, bit_of(l[k]));
        }
        if (do_tt) {
          group_place<D, TV, LB>(g, facet_key<D, 1>(l), s, 1, M.err);
          group_place<D, TV, LB>(g, facet_key<D, 2>(l), s, 2, M.err);
          if constexpr (D == 4) group_place<D, TV, LB>(g, facet_key<D, 3>(l), s, 3, M.err);
        }
      }
    }
  }
  __syncthreads();

  // ---- P4: A joins the facets 0 of the simplices (x, p, ..); B expands VV row p ----------------
  int n_vv = 0;
  if (!isB) {
    if (do_tt && live) {
      GroupCtx g;
      const int hs = C.hs;
      g.tbl = tbl + p;
      g.hs = (uint32_t)hs;
      g.ttrow = ttrow;
      g.tets = tets; g.texid = texid; g.gid = gid; g.tt = O.tt_indices;
      g.t_lo = t_lo; g.tt_slot = ctx->tt_slot; g.c_lo = td.v_lo - td.row_rel; g.c_tlo = t_lo - td.tt_rel;
      g.s_ext = s_ext; g.s_all = S;
      // the flagged entries among the first 32 come from the walk's mask, longer rows are scanned for the rest
      for (uint32_t fm = fmask; fm != 0u; fm &= fm - 1u) {
        const int s = (int)(st_vt[off + __ffs(fm) - 1] & 0x7FFFu);
        int l[4];
        load_local<LB>(tets, s, l);
        group_place<D, TV, LB>(g, facet_key<D, 0>(l), s, 0, M.err);
      }
      int i = off + 32;
      const int end = off + nb;
      for (;;) {
        uint32_t e = 0u;
        while (i < end && !((e = st_vt[i]) & 0x8000u)) ++i;
        if (i >= end) break;
        ++i;
        const int s = (int)(e & 0x7FFFu);
        int l[4];
        load_local<LB>(tets, s, l);
        group_place<D, TV, LB>(g, facet_key<D, 0>(l), s, 0, M.err);
      }
    }
  } else if (do_vv) {
    const int wV = (td.nloc + 31) >> 5;
    uint32_t* row = bmV + p;
    int nbv = 0;
    if (live) {
      // (p itself is never marked: a vertex is not its own neighbour)
#pragma unroll 4
      for (int w = 0; w < wV; ++w) nbv += __popc(row[w * TV]);
    }
    uint32_t tot;
    const int offv = (int)half_exclusive_scan<NT>((uint32_t)nbv, scan, &tot);
    if (tid == TV) scan[34] = tot;
    if (live) {
      O.vv_offsets[row0 + p] = vv0 + offv;
      int pos = offv, lbase = -32;
      uint32_t bits = 0u;
      for (int n = 0; n < nbv; ++n) {
        while (bits == 0u) { bits = *row; row += TV; lbase += 32; }
        if (GALE_IN_BOUNDS(M.err, pos >= 0 && pos < C.vv_max && lbase + __ffs(bits) - 1 < td.nloc))
          st_vv[pos++] = (uint16_t)(lbase + __ffs(bits) - 1);
        bits &= bits - 1;
      }
    }
  }
  __syncthreads();
  n_vv = (int)scan[34];
  if (tid == 0 && ((do_vt && n_vt != td.vt_nnz) || (do_vv && n_vv != td.vv_nnz)))
    raise_err(M.err, ERR_SIZE_MISMATCH);  // the sizes fixed at create must be reproduced exactly

  // ---- P5: translate to global ids, coalesced write-out ----------------------------------------
  if (do_tt) {
    const int c_lo = td.v_lo - td.row_rel, c_hi = c_lo + td.c_rows;  // the cluster's vertex range
    for (int i = tid; i < s_int; i += NT) {
      bool need_fb = false;
      {
        uint32_t e[D];
        if constexpr (D == 4) {
          const uint2 q = reinterpret_cast<const uint2*>(ttrow)[i];
          e[0] = q.x & 0xFFFFu; e[1] = q.x >> 16; e[2] = q.y & 0xFFFFu; e[3] = q.y >> 16;
        } else {
          e[0] = ttrow[i * 3]; e[1] = ttrow[i * 3 + 1]; e[2] = ttrow[i * 3 + 2];
        }
        int r[D];
#pragma unroll
        for (int k = 0; k < D; ++k)
          r[k] = e[k] == 0xFFFFu ? -1 : ((int)e[k] < s_ext ? texid[e[k]] : t_lo + ((int)e[k] - s_ext));
        bool delegated = false;
        if (r[0] < 0) {
          int l[4];
          load_local<LB>(tets, s_ext + i, l);
          // facet 0 = (l[1], ..) has no vertex in this tile when l[1] lies above it: the tile that owns l[1]
          // writes the entry if it belongs to this cluster, else it is resolved from global memory (a5)
          const bool out0 = l[1] - nlo >= nrows;
          delegated = out0 && gid[l[1]] < c_hi;
          need_fb = out0 && !delegated;
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
          if (!delegated) o[0] = r[0];
          o[1] = r[1]; o[2] = r[2];
        }
      }
      if (need_fb) {  // rare (cross-cluster facets only): a plain atomic per facet
        const uint32_t pos = atomicAdd(&scan[33], 1u);
        if (GALE_IN_BOUNDS(M.err, (int)pos < C.sint)) fbq[pos] = (uint16_t)i;
      }
    }
  }
  if (do_vt)
    for (int i = tid; i < n_vt; i += NT) {
      const int s = (int)(st_vt[i] & 0x7FFFu);
      GALE_ST(O.vt_indices + vt0 + i, s < s_ext ? texid[s] : t_lo + (s - s_ext));
    }
  if (do_vv)
    for (int i = tid; i < n_vv; i += NT) GALE_ST(O.vv_indices + vv0 + i, gid[st_vv[i]]);

  if (do_tt) {
    __syncthreads();  // queue complete, TT rows stored
    // ---- a5: one queued facet per thread, resolved from global memory -------------------------
    const int nq = (int)scan[33];
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
}

}  // namespace gale
