// gale_lib.cu — C-ABI boundary of the GALE relation hot path (include/gale.h).
//
// Host side of the paper's producer: initialization (I_T, T_ex, interval arrays),
// the leader producer's batch set-up and launch and the bounded queue of
// pre-allocated result buffers handed to consumers. Every relation entry is
// computed by the kernels in gale_kernels.cuh; nothing here computes VT/VV/TT on the CPU.
#include "gale_kernels.cuh"
#include "gale_walk.cuh"

#include <algorithm>
#include <atomic>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <memory>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

#include "../../include/gale.h"

namespace {

using gale::DeviceMesh;
using gale::SmemCfg;
using gale::TileDesc;

thread_local std::string g_last_error;

#define GALE_CUDA(call)                                                                                  \
  do {                                                                                                   \
    cudaError_t e_ = (call);                                                                             \
    if (e_ != cudaSuccess) {                                                                             \
      g_last_error = std::string(#call) + ": " + cudaGetErrorString(e_);                                 \
      return GALE_ERR_CUDA;                                                                              \
    }                                                                                                    \
  } while (0)

constexpr size_t kAlign = 256;
inline size_t up(size_t x, size_t a = kAlign) { return (x + a - 1) / a * a; }
inline long long pad_to(long long x, long long a) { return (x + a - 1) / a * a; }
constexpr int kSmemLimit = 227 * 1024;  // opt-in dynamic shared memory per block on sm_100

// ---- result of the create-time analysis ----------------------------------------------------------
struct Plan {
  // key
  const int32_t* dT = nullptr;
  int dim = 0, nV = 0, nC = 0, tv_req = 0, maxB = 1, queue_depth = 0, device_ring = 0;
  long long nT = 0;
  uint32_t flags = 0;
  std::vector<int32_t> cl_off;
  // index (host copies)
  int tv = 0, nTiles = 0, NT = 0;
  std::vector<int32_t> first_tet, opp_first, opp_perm, cl_tile_begin, tex, gid;
  std::vector<uint16_t> loc;            // 4 per staged simplex (build); compacted into loc8 when lb == 1
  std::vector<uint8_t> loc8;
  long long staged_padded = 0;          // staged simplices incl. per-tile padding
  std::vector<TileDesc> tiles;
  SmemCfg cfg{};                        // capacities for the full relation mask
  int smem_bytes = 0;
  // the walk kernel (gale_walk.cuh) on the same tiles: same capacities + per-vertex table size
  int gmax = 1;                         // largest facet group of a vertex
  int w_NT = 0, w_smem = 0;
  bool walk_ok = false;
  long long ext_refs = 0, vt_total = 0, vv_total = 0;
  // per-cluster sizes
  std::vector<long long> cl_vt, cl_vv;  // nnz per cluster
  std::vector<int32_t> cl_t_lo;         // [nC+1] first internal simplex of cluster c (I_T)
  long long max_rows = 0, max_vt = 0, max_vv = 0, max_tt = 0;
  double analyse_ms = 0;

};

struct SlotLayout {
  size_t vt_off = 0, vt_idx = 0, vv_off = 0, vv_idx = 0, tt = 0, total = 0;
};
SlotLayout slot_capacity_layout(const Plan& p, int maxB) {
  const int D = p.dim + 1;
  SlotLayout L;
  size_t o = 0;
  L.vt_off = o; o = up(o + (size_t(maxB) * p.max_rows + 1) * 4);
  L.vt_idx = o; o = up(o + size_t(maxB) * p.max_vt * 4);
  L.vv_off = o; o = up(o + (size_t(maxB) * p.max_rows + 1) * 4);
  L.vv_idx = o; o = up(o + size_t(maxB) * p.max_vv * 4);
  L.tt = o;     o = up(o + size_t(maxB) * p.max_tt * D * 4);
  L.total = o;
  return L;
}

int validate_host(const Plan& p, const std::vector<int32_t>& T) {
  const int D = p.dim + 1;
  for (long long t = 0; t < p.nT; ++t) {
    const int32_t* r = T.data() + t * D;
    if (r[0] < 0 || r[D - 1] >= p.nV) return GALE_ERR_NOT_CANONICAL;
    for (int k = 1; k < D; ++k)
      if (r[k] <= r[k - 1]) return GALE_ERR_NOT_CANONICAL;
    if (t > 0 && !std::lexicographical_compare(r - D, r, r, r + D)) return GALE_ERR_NOT_CANONICAL;
  }
  return GALE_OK;
}

// C4: every facet has at most two cofaces (sorted facet list, like the paper's sorted F list, :178).
template <int D>
int validate_manifold(const Plan& p, const std::vector<int32_t>& T) {
  struct F { int32_t v[D - 1]; };
  std::vector<F> f(size_t(p.nT) * D);
  for (long long t = 0; t < p.nT; ++t)
    for (int k = 0; k < D; ++k) {
      int o = 0;
      for (int j = 0; j < D; ++j)
        if (j != k) f[t * D + k].v[o++] = T[t * D + j];
    }
  auto less = [](const F& a, const F& b) { return std::lexicographical_compare(a.v, a.v + D - 1, b.v, b.v + D - 1); };
  std::sort(f.begin(), f.end(), less);
  for (size_t i = 2; i < f.size(); ++i)
    if (!less(f[i - 2], f[i])) return GALE_ERR_NONMANIFOLD;
  return GALE_OK;
}

inline int threads_for_tile(int tv) {  // NT >= tv (one thread per row in P2)
  if (const char* e = std::getenv("GALE_NT")) { const int v = std::atoi(e); if ((v == 128 || v == 256) && v >= tv) return v; }
  return tv > 128 ? 256 : 128;
}

// Kernel capacities for one launch: regions the relation mask does not need are dropped.
SmemCfg cfg_for_mask(const SmemCfg& full, uint32_t mask, bool count_mode) {
  SmemCfg c = full;
  if (!(mask & gale::REL_VV)) { c.WV = 0; c.vv_max = 0; }
  if (!(mask & gale::REL_TT) || count_mode) { c.tbl = 0; c.sint = 0; }
  if (!(mask & gale::REL_VT)) c.vt_max = 0;
  if (count_mode) { c.vt_max = 0; c.vv_max = 0; c.sext = 0; c.nloc = 0; }  // T_ex ids / vertex table are not staged
  return c;
}

inline gale::SmemLayout layout_for(int D, const SmemCfg& c) {
  return D == 4 ? gale::make_layout<4>(c) : gale::make_layout<3>(c);
}

using KernelFn = void (*)(const DeviceMesh, const gale::BatchParams, const SmemCfg, const gale::SmemLayout,
                          const gale::OutPtrs);
template <int D, bool COUNT, int LB>
KernelFn kernel_for_nt(int NT) {
  return NT == 256 ? gale::gale_batch_kernel<D, 256, COUNT, LB> : gale::gale_batch_kernel<D, 128, COUNT, LB>;
}
template <int D, bool COUNT>
KernelFn kernel_for_lb(int NT, int lb) { return lb == 1 ? kernel_for_nt<D, COUNT, 1>(NT) : kernel_for_nt<D, COUNT, 2>(NT); }
KernelFn kernel_for(int D, int NT, bool count, int lb) {
  if (D == 4) return count ? kernel_for_lb<4, true>(NT, lb) : kernel_for_lb<4, false>(NT, lb);
  return count ? kernel_for_lb<3, true>(NT, lb) : kernel_for_lb<3, false>(NT, lb);
}

using WalkFn = void (*)(const DeviceMesh, const gale::BatchParams, const SmemCfg, const gale::WalkLayout, const gale::OutPtrs);
template <int D, int LB>
WalkFn walk_for_nt(int NT) {
  return NT == 512 ? gale::gale_walk_kernel<D, 512, LB>
                   : (NT == 256 ? gale::gale_walk_kernel<D, 256, LB>
                                : (NT == 128 ? gale::gale_walk_kernel<D, 128, LB> : gale::gale_walk_kernel<D, 64, LB>));
}
WalkFn walk_kernel_for(int D, int NT, int lb) {
  if (D == 4) return lb == 1 ? walk_for_nt<4, 1>(NT) : walk_for_nt<4, 2>(NT);
  return lb == 1 ? walk_for_nt<3, 1>(NT) : walk_for_nt<3, 2>(NT);
}
inline int walk_threads_for_tile(int tv) { return tv > 128 ? 512 : (tv > 64 ? 256 : (tv > 32 ? 128 : 64)); }  // NT = 2 * rows
SmemCfg walk_cfg_for_mask(const SmemCfg& full, uint32_t mask) {
  SmemCfg c = full;
  c.tbl = 0;
  if (!(mask & gale::REL_VV)) { c.WV = 0; c.vv_max = 0; }
  if (!(mask & gale::REL_TT)) { c.hs = 0; c.sint = 0; }
  if (!(mask & (gale::REL_VT | gale::REL_TT))) c.vt_max = 0;  // TT reads the staged VT entries' flags
  return c;
}
inline gale::WalkLayout walk_layout_for(int D, const SmemCfg& c) {
  return D == 4 ? gale::make_walk_layout<4>(c) : gale::make_walk_layout<3>(c);
}

// The dynamic shared-memory ceiling is an attribute of the kernel instantiation for the whole context,
// not of a handle: raise every instantiation to the device limit once, never lower it.
cudaError_t allow_max_smem(KernelFn fn) { return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit); }

// Tiles of `tv` vertices, their T_ex lists, halo lists and the tile-local encoding of their staged
// simplices. Returns false if a tile exceeds a kernel limit for this tv (the caller retries smaller).
bool build_tiles(Plan& p, const std::vector<int32_t>& T, int tv) {
  const int D = p.dim + 1;
  p.tv = tv;
  p.NT = threads_for_tile(tv);
  std::vector<int32_t> tile_vlo;
  p.cl_tile_begin.assign(p.nC + 1, 0);
  for (int c = 0; c < p.nC; ++c) {
    p.cl_tile_begin[c] = int(tile_vlo.size());
    for (int v = p.cl_off[c]; v < p.cl_off[c + 1]; v += tv) tile_vlo.push_back(v);
  }
  p.cl_tile_begin[p.nC] = int(tile_vlo.size());
  p.nTiles = int(tile_vlo.size());
  tile_vlo.push_back(p.nV);
  const int nTiles = p.nTiles;
  std::vector<int32_t> tile_of(p.nV), tile_vhi(nTiles);
  for (int c = 0; c < p.nC; ++c)
    for (int i = p.cl_tile_begin[c]; i < p.cl_tile_begin[c + 1]; ++i) {
      tile_vhi[i] = std::min(tile_vlo[i] + tv, p.cl_off[c + 1]);
      for (int v = tile_vlo[i]; v < tile_vhi[i]; ++v) tile_of[v] = i;
    }
  // T_ex: simplex t is external to every tile it touches other than the tile of its lowest vertex
  std::vector<long long> raw_off(nTiles + 1, 0);
  std::vector<int32_t> raw;
  for (int pass = 0; pass < 2; ++pass) {
    std::vector<long long> cur;
    if (pass == 1) {
      for (int i = 0; i < nTiles; ++i) raw_off[i + 1] += raw_off[i];
      raw.resize(size_t(raw_off[nTiles]));
      cur.assign(raw_off.begin(), raw_off.end() - 1);
    }
    for (long long t = 0; t < p.nT; ++t) {
      const int32_t* r = T.data() + t * D;
      const int t0 = tile_of[r[0]];
      int seen[3], ns = 0;
      for (int k = 1; k < D; ++k) {
        const int tk = tile_of[r[k]];
        if (tk == t0) continue;
        bool dup = false;
        for (int s = 0; s < ns; ++s) dup |= seen[s] == tk;
        if (dup) continue;
        seen[ns++] = tk;
        if (pass == 0) ++raw_off[tk + 1]; else raw[size_t(cur[tk]++)] = int32_t(t);
      }
    }
  }
  p.ext_refs = raw_off[nTiles];
  // descriptors, padded offsets, limits that need no halo
  p.tiles.assign(nTiles, TileDesc{});
  long long stg = 0, texo = 0;
  const int max_local = D == 4 ? gale::kMaxLocal4 : gale::kMaxLocal3;
  for (int c = 0; c < p.nC; ++c)
    for (int i = p.cl_tile_begin[c]; i < p.cl_tile_begin[c + 1]; ++i) {
      TileDesc& d = p.tiles[i];
      d.v_lo = tile_vlo[i];
      d.nrows = tile_vhi[i] - tile_vlo[i];
      d.t_lo = p.first_tet[d.v_lo];
      d.s_int = p.first_tet[tile_vhi[i]] - d.t_lo;
      d.s_ext = int(raw_off[i + 1] - raw_off[i]);
      d.row_rel = d.v_lo - p.cl_off[c];
      d.c_rows = p.cl_off[c + 1] - p.cl_off[c];
      d.tt_rel = d.t_lo - p.first_tet[p.cl_off[c]];
      d.stg_off = stg;
      d.tex_off = texo;
      const long long S = (long long)d.s_int + d.s_ext;
      if (S > (D == 4 ? gale::kMaxStaged4 : gale::kMaxStaged3)) return false;
      stg += pad_to(S, 4);
      texo += pad_to(d.s_ext, 4);
    }
  p.staged_padded = stg;
  p.loc.assign(size_t(stg) * 4 + 16, 0);
  p.loc8.clear();
  p.tex.assign(size_t(texo) + 4, 0);
  for (int i = 0; i < nTiles; ++i)
    std::copy(raw.begin() + raw_off[i], raw.begin() + raw_off[i + 1], p.tex.begin() + p.tiles[i].tex_off);
  // halo + local encoding, tiles split over host threads
  const int nth = std::max(1, std::min<int>(32, std::min<int>(int(std::thread::hardware_concurrency()), nTiles / 64 + 1)));
  std::vector<std::vector<int32_t>> gid_part(nth);
  std::vector<int> tile_lo(nth + 1);
  for (int w = 0; w <= nth; ++w) tile_lo[w] = int((long long)nTiles * w / nth);
  std::atomic<bool> ok{true};
  auto work = [&](int w) {
    std::vector<uint16_t> map(size_t(p.nV), uint16_t(0xFFFF));
    std::vector<int32_t>& hp = gid_part[w];
    std::vector<int32_t> h;
    for (int i = tile_lo[w]; i < tile_lo[w + 1] && ok.load(std::memory_order_relaxed); ++i) {
      TileDesc& d = p.tiles[i];
      const int v_lo = d.v_lo, v_hi = d.v_lo + d.nrows;
      const int32_t* ex = p.tex.data() + d.tex_off;
      auto simplex = [&](int s) { return T.data() + (long long)(s < d.s_ext ? ex[s] : d.t_lo + (s - d.s_ext)) * D; };
      const int S = d.s_int + d.s_ext;
      h.clear();
      for (int s = 0; s < S; ++s) {
        const int32_t* r = simplex(s);
        for (int k = 0; k < D; ++k)
          if ((r[k] < v_lo || r[k] >= v_hi) && map[r[k]] == 0xFFFF) { map[r[k]] = 0xFFFE; h.push_back(r[k]); }
      }
      std::sort(h.begin(), h.end());
      const int nhalo = int(h.size());
      const int nlo = int(std::lower_bound(h.begin(), h.end(), v_lo) - h.begin());
      if (nhalo + d.nrows > max_local) {
        for (int v : h) map[v] = 0xFFFF;
        ok.store(false);
        return;
      }
      for (int j = 0; j < nhalo; ++j) map[h[j]] = uint16_t(j < nlo ? j : j + d.nrows);
      d.nlo = nlo;
      d.nloc = nhalo + d.nrows;
      d.gid_off = (long long)hp.size();  // relative to this thread's part; rebased below
      uint16_t* out = p.loc.data() + d.stg_off * 4;
      for (int s = 0; s < S; ++s) {
        const int32_t* r = simplex(s);
        for (int k = 0; k < 4; ++k)
          out[s * 4 + k] = k >= D ? uint16_t(0xFFFF)
                                  : (r[k] >= v_lo && r[k] < v_hi) ? uint16_t(nlo + (r[k] - v_lo)) : map[r[k]];
      }
      hp.insert(hp.end(), h.begin(), h.begin() + nlo);  // local id -> global id, ascending
      for (int v = v_lo; v < v_hi; ++v) hp.push_back(v);
      hp.insert(hp.end(), h.begin() + nlo, h.end());
      hp.resize(size_t(pad_to((long long)hp.size(), 4)), 0);
      for (int v : h) map[v] = 0xFFFF;
    }
  };
  {
    std::vector<std::thread> th;
    for (int w = 1; w < nth; ++w) th.emplace_back(work, w);
    work(0);
    for (auto& t : th) t.join();
  }
  if (!ok.load()) return false;
  long long hoff = 0;
  for (int w = 0; w < nth; ++w) {
    for (int i = tile_lo[w]; i < tile_lo[w + 1]; ++i) p.tiles[i].gid_off += hoff;
    hoff += (long long)gid_part[w].size();
  }
  p.gid.assign(size_t(hoff) + 4, 0);
  hoff = 0;
  for (int w = 0; w < nth; ++w) {
    std::copy(gid_part[w].begin(), gid_part[w].end(), p.gid.begin() + hoff);
    hoff += (long long)gid_part[w].size();
    std::vector<int32_t>().swap(gid_part[w]);
  }
  // largest facet group of a tile vertex (walk kernel's private tables): D-1 facets per simplex of its
  // run + facet 0 of every simplex whose second vertex it is
  p.gmax = 1;
  for (int v = 0; v < p.nV; ++v)
    p.gmax = std::max(p.gmax, (D - 1) * (p.first_tet[v + 1] - p.first_tet[v]) + (p.opp_first[v + 1] - p.opp_first[v]));
  // shared-memory capacities known so far
  long long smax = 4, sext = 4, sint = 2, nloc = 4;
  for (const TileDesc& d : p.tiles) {
    smax = std::max(smax, pad_to((long long)d.s_int + d.s_ext, 4));
    sext = std::max(sext, pad_to(d.s_ext, 4));
    sint = std::max(sint, pad_to(d.s_int, 2));
    nloc = std::max(nloc, pad_to(d.nloc, 4));
  }
  p.cfg = SmemCfg{};
  p.cfg.tv = tv;
  p.cfg.smax = int(smax);
  p.cfg.sext = int(sext);
  p.cfg.nloc = int(nloc);
  // 8-bit local ids when every tile has at most 255 local vertices: half the staged bytes (HBM and
  // shared memory). 0xFF only pads the unused 4th entry of a triangle.
  p.cfg.lb = nloc <= 255 ? 1 : 2;
  if (p.cfg.lb == 1) {
    p.loc8.resize(p.loc.size());
    for (size_t i = 0; i < p.loc.size(); ++i) p.loc8[i] = uint8_t(p.loc[i]);
    std::vector<uint16_t>().swap(p.loc);
  }
  p.cfg.sint = int(sint);
  p.cfg.WT = int((smax + 31) / 32) | 1;
  p.cfg.WV = int((nloc + 31) / 32) | 1;
  return true;
}

struct DevBuf {  // temporary device memory of the analysis
  void* p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
  int alloc(size_t n) { GALE_CUDA(cudaMalloc(&p, std::max<size_t>(n, 16))); return GALE_OK; }
  template <class V>
  int upload(const V& v, cudaStream_t st) {
    int rc = alloc(v.size() * sizeof(typename V::value_type));
    if (rc != GALE_OK) return rc;
    if (!v.empty())
      GALE_CUDA(cudaMemcpyAsync(p, v.data(), v.size() * sizeof(typename V::value_type), cudaMemcpyHostToDevice, st));
    return GALE_OK;
  }
};

// Sizing run (count mode of the batch kernel) over all tiles: exact VT / VV entry counts per tile.
// `fits` tells whether the count-mode shared memory fits at this tile size.
int run_sizing(Plan& p, const int32_t* dT, cudaStream_t st, std::vector<long long>& stats, bool& fits) {
  const int D = p.dim + 1;
  fits = true;
  stats.assign(size_t(p.nTiles) * 4, 0);
  if (p.nTiles == 0) return GALE_OK;
  const SmemCfg full = p.cfg;
  const std::vector<uint32_t> parts = {3u};
  if (layout_for(D, cfg_for_mask(full, 3, true)).total > kSmemLimit) { fits = false; return GALE_OK; }

  DevBuf b_ft, b_tiles, b_tex, b_gid, b_loc, b_stats, b_err;
  int rc;
  if ((rc = b_ft.upload(p.first_tet, st)) || (rc = b_tiles.upload(p.tiles, st)) || (rc = b_tex.upload(p.tex, st)) ||
      (rc = b_gid.upload(p.gid, st)) || (rc = (p.cfg.lb == 1 ? b_loc.upload(p.loc8, st) : b_loc.upload(p.loc, st))) ||
      (rc = b_stats.alloc(stats.size() * 8)) || (rc = b_err.alloc(4)))
    return rc;
  GALE_CUDA(cudaMemsetAsync(b_err.p, 0, 4, st));
  DeviceMesh dm{};
  dm.T = dT;
  dm.first_tet = static_cast<int32_t*>(b_ft.p);
  dm.tiles = static_cast<TileDesc*>(b_tiles.p);
  dm.tex = static_cast<int32_t*>(b_tex.p);
  dm.gid = static_cast<int32_t*>(b_gid.p);
  dm.loc = b_loc.p;
  dm.err = static_cast<int32_t*>(b_err.p);
  KernelFn fn = kernel_for(D, p.NT, true, p.cfg.lb);
  std::vector<long long> part_stats(stats.size());
  for (uint32_t m : parts) {
    const SmemCfg c = cfg_for_mask(full, m, true);
    const gale::SmemLayout lay = layout_for(D, c);
    const int smem = lay.total;
    GALE_CUDA(allow_max_smem(fn));
    gale::BatchParams P{};
    P.mask = m | gale::MODE_COUNT;
    gale::OutPtrs O{};
    O.stats = static_cast<long long*>(b_stats.p);
    fn<<<p.nTiles, p.NT, smem, st>>>(dm, P, c, lay, O);
    GALE_CUDA(cudaGetLastError());
    GALE_CUDA(cudaMemcpyAsync(part_stats.data(), b_stats.p, stats.size() * 8, cudaMemcpyDeviceToHost, st));
    GALE_CUDA(cudaStreamSynchronize(st));
    for (int i = 0; i < p.nTiles; ++i) {
      if (m & 1) stats[i * 4 + 0] = part_stats[i * 4 + 0];
      if (m & 2) stats[i * 4 + 1] = part_stats[i * 4 + 1];
    }
  }
  int err = 0;
  GALE_CUDA(cudaMemcpyAsync(&err, b_err.p, 4, cudaMemcpyDeviceToHost, st));
  GALE_CUDA(cudaStreamSynchronize(st));
  if (err) { g_last_error = "device guard fired during sizing: " + std::to_string(err); return GALE_ERR_WORKSPACE; }
  return GALE_OK;
}

int analyse(const gale_mesh_desc_t& d, cudaStream_t st, std::unique_ptr<Plan>& out) {
  const auto t0 = std::chrono::steady_clock::now();
  auto p = std::make_unique<Plan>();
  p->dT = d.d_simplices; p->dim = d.dim; p->nV = d.num_vertices; p->nC = d.num_clusters; p->nT = d.num_simplices;
  p->tv_req = d.tile_vertices; p->flags = d.flags;
  p->maxB = d.max_batch_clusters; p->queue_depth = d.queue_depth; p->device_ring = d.device_ring;
  p->cl_off.assign(d.h_cluster_offsets, d.h_cluster_offsets + d.num_clusters + 1);
  const int D = d.dim + 1;
  if (p->cl_off.front() != 0 || p->cl_off.back() != p->nV) return GALE_ERR_INVALID_ARG;
  for (int c = 0; c < p->nC; ++c)
    if (p->cl_off[c] > p->cl_off[c + 1]) return GALE_ERR_INVALID_ARG;

  std::vector<int32_t> T(size_t(p->nT) * D);
  if (p->nT) GALE_CUDA(cudaMemcpy(T.data(), d.d_simplices, T.size() * 4, cudaMemcpyDeviceToHost));
  if (d.flags & (GALE_VALIDATE | GALE_VALIDATE_MANIFOLD)) {
    int rc = validate_host(*p, T);
    if (rc != GALE_OK) return rc;
  }
  if (d.flags & GALE_VALIDATE_MANIFOLD) {
    int rc = D == 4 ? validate_manifold<4>(*p, T) : validate_manifold<3>(*p, T);
    if (rc != GALE_OK) return rc;
  }
  // I_T: first simplex whose lowest vertex is >= v; and the same keyed by the second vertex
  p->first_tet.assign(p->nV + 1, 0);
  p->opp_first.assign(p->nV + 1, 0);
  for (long long t = 0; t < p->nT; ++t) {
    ++p->first_tet[T[t * D] + 1];
    ++p->opp_first[T[t * D + 1] + 1];
  }
  for (int v = 0; v < p->nV; ++v) {
    p->first_tet[v + 1] += p->first_tet[v];
    p->opp_first[v + 1] += p->opp_first[v];
  }
  p->opp_perm.resize(size_t(p->nT));
  {
    std::vector<int32_t> cur(p->opp_first.begin(), p->opp_first.end() - 1);
    for (long long t = 0; t < p->nT; ++t) p->opp_perm[cur[T[t * D + 1]]++] = int32_t(t);
  }
  p->cl_t_lo.resize(p->nC + 1);
  for (int c = 0; c <= p->nC; ++c) p->cl_t_lo[c] = p->first_tet[p->cl_off[c]];

  int tv = d.tile_vertices > 0 ? std::min(d.tile_vertices, gale::kMaxTileVertices) : (d.dim == 3 ? 32 : 64);  // measured optima on configs 5 and 2 (profiles/r1_v5_ncu_summary.md)
  std::vector<long long> stats;
  bool shrunk = false;
  for (;; tv = (tv + 1) / 2) {
    if (tv < 1) return GALE_ERR_UNSUPPORTED;
    const bool last = tv == 1;
    bool fits = build_tiles(*p, T, tv);
    if (fits) {
      int rc = run_sizing(*p, d.d_simplices, st, stats, fits);
      if (rc != GALE_OK) return rc;
    }
    if (fits) {
      long long vt_max = 1, vv_max = 1, tbl_max = 4;
      for (int i = 0; i < p->nTiles; ++i) {
        vt_max = std::max(vt_max, stats[i * 4 + 0]);
        vv_max = std::max(vv_max, stats[i * 4 + 1]);
        tbl_max = std::max(tbl_max, stats[i * 4 + 0] + (long long)(D - 2) * p->tiles[i].s_int);
      }
      p->cfg.vt_max = int(pad_to(vt_max, 8));
      p->cfg.vv_max = int(pad_to(vv_max, 8));
      p->cfg.tbl = int(pad_to(tbl_max, 4));
      p->smem_bytes = layout_for(D, p->cfg).total;
      fits = vt_max <= gale::kMaxNnz16 && vv_max <= gale::kMaxNnz16 && p->smem_bytes <= kSmemLimit;
    }
    // automatic tile size: tiles whose vertices are scattered in the mesh (graded meshes, config 4) need
    // large per-block capacities and leave few resident blocks; half the tile measured +25 % there
    if (fits && d.tile_vertices == 0 && !shrunk && tv >= 32 && D == 4 && p->smem_bytes > 56 * 1024) {
      shrunk = true;
      continue;
    }
    if (fits) break;
    if (last) { g_last_error = "a single vertex star exceeds the kernel's shared-memory limits"; return GALE_ERR_UNSUPPORTED; }
  }
  {  // can the walk kernel run these tiles?
    // load <= 3/4 even if no facet of a group is shared; every interior facet is recorded twice, so the
    // usual load is about 0.4 (measured: at 0.54 the re-probes cost 3 warp-instructions per tet)
    p->cfg.hs = std::max(8, (p->gmax + p->gmax / 3 + 1) & ~1);
    p->w_NT = walk_threads_for_tile(p->tv);
    p->w_smem = walk_layout_for(D, walk_cfg_for_mask(p->cfg, 7)).total;
    p->walk_ok = p->tv <= 256 && p->w_smem <= kSmemLimit && p->cfg.smax < 32768 && p->cfg.vt_max < 65536;
  }
  // per-tile output placement inside its cluster, per-cluster sizes
  p->cl_vt.assign(p->nC, 0);
  p->cl_vv.assign(p->nC, 0);
  for (int c = 0; c < p->nC; ++c) {
    long long vt = 0, vv = 0;
    for (int i = p->cl_tile_begin[c]; i < p->cl_tile_begin[c + 1]; ++i) {
      TileDesc& t = p->tiles[i];
      if (vt > INT32_MAX || vv > INT32_MAX) return GALE_ERR_UNSUPPORTED;
      t.vt_rel = int32_t(vt); t.vv_rel = int32_t(vv);
      t.vt_nnz = int32_t(stats[i * 4 + 0]); t.vv_nnz = int32_t(stats[i * 4 + 1]);
      vt += t.vt_nnz; vv += t.vv_nnz;
    }
    p->cl_vt[c] = vt; p->cl_vv[c] = vv;
    p->vt_total += vt; p->vv_total += vv;
    p->max_rows = std::max<long long>(p->max_rows, p->cl_off[c + 1] - p->cl_off[c]);
    p->max_vt = std::max(p->max_vt, vt);
    p->max_vv = std::max(p->max_vv, vv);
    p->max_tt = std::max<long long>(p->max_tt, p->cl_t_lo[c + 1] - p->cl_t_lo[c]);
  }
  p->analyse_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  out = std::move(p);
  return GALE_OK;
}

int check_desc(const gale_mesh_desc_t* d) {
  if (!d || (d->dim != 2 && d->dim != 3) || d->num_vertices < 0 || d->num_simplices < 0 || d->num_clusters < 0 ||
      !d->h_cluster_offsets || (d->num_simplices > 0 && !d->d_simplices) || d->max_batch_clusters < 1 ||
      d->queue_depth < 0 || d->device_ring < 0 || d->tile_vertices < 0 || d->num_simplices >= (1LL << 31) - 1 ||
      (d->flags & ~uint32_t(GALE_VALIDATE | GALE_VALIDATE_MANIFOLD | GALE_STREAM_ORDERED | GALE_KERNEL_DENSE | GALE_KERNEL_WALK)) ||
      (d->flags & (GALE_KERNEL_DENSE | GALE_KERNEL_WALK)) == (GALE_KERNEL_DENSE | GALE_KERNEL_WALK))
    return GALE_ERR_INVALID_ARG;
  if (reinterpret_cast<uintptr_t>(d->d_simplices) % 16) return GALE_ERR_INVALID_ARG;
  return GALE_OK;
}
int check_device() {
  int dev = 0;
  cudaDeviceProp prop{};
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    cudaGetLastError();
    g_last_error = "no CUDA device";
    return GALE_ERR_UNSUPPORTED;
  }
  if (prop.major != 10) {
    g_last_error = "device is not sm_100 (compute capability " + std::to_string(prop.major) + "." + std::to_string(prop.minor) + ")";
    return GALE_ERR_UNSUPPORTED;
  }
  return GALE_OK;
}

// Placement of the index arrays inside the caller's workspace: ONE function serves both the size
// query and the upload, so the two cannot disagree.
struct IndexLayout {
  size_t first_tet = 0, opp_first = 0, opp_perm = 0, cl_tile_begin = 0, tiles = 0, tex = 0, gid = 0, loc = 0, total = 0;
};
IndexLayout index_layout(const Plan& p) {
  IndexLayout L;
  size_t o = 0;
  auto take = [&](size_t bytes) { const size_t at = o; o = up(o + bytes + 64); return at; };  // 64: vector loads may read past the end
  L.first_tet = take(p.first_tet.size() * 4);
  L.opp_first = take(p.opp_first.size() * 4);
  L.opp_perm = take(p.opp_perm.size() * 4);
  L.cl_tile_begin = take(p.cl_tile_begin.size() * 4);
  L.tiles = take(p.tiles.size() * sizeof(TileDesc));
  L.tex = take(p.tex.size() * 4);
  L.gid = take(p.gid.size() * 4);
  L.loc = take(p.cfg.lb == 1 ? p.loc8.size() : p.loc.size() * 2);
  L.total = o;
  return L;
}
int slots_of(int queue_depth, int device_ring) { return queue_depth > 0 ? queue_depth : (device_ring > 0 ? device_ring : 4); }
size_t total_workspace(const Plan& p) {
  return index_layout(p).total + size_t(slots_of(p.queue_depth, p.device_ring)) * slot_capacity_layout(p, p.maxB).total;
}

enum SlotState { SLOT_FREE = 0, SLOT_SUBMITTED = 1, SLOT_POPPED = 2 };

struct Slot {
  char* dev = nullptr;
  char* pinned = nullptr;
  cudaEvent_t ev_submit = nullptr, ev_start = nullptr, ev_done = nullptr, ev_ready = nullptr;
  std::atomic<int> state{SLOT_FREE};
  long long seq = 0;
  int n = 0;
  uint32_t mask = 0;
  std::vector<int32_t> ids, row_begin, tt_row_begin;
  long long rows = 0, vt_nnz = 0, vv_nnz = 0, tt_rows = 0;
  SlotLayout used;  // section offsets of this batch
  float prep_ms = 0.f;
  std::chrono::steady_clock::time_point t_submit;
};

}  // namespace

struct gale_plan {
  std::unique_ptr<Plan> plan;
};

struct gale_mesh {
  std::unique_ptr<Plan> plan;
  int dim = 0, D = 0, maxB = 0, queue_depth = 0;
  bool stream_ordered = false;
  int kernel = 0;  // 0 = dense kernel (gale_kernels.cuh), 1 = walk kernel (gale_walk.cuh)
  DeviceMesh dm{};
  std::vector<std::unique_ptr<Slot>> slots;
  SlotLayout cap;
  cudaStream_t side = nullptr;
  // Consecutive batches are launched in turn on these library-owned streams, each ordered after the
  // caller's stream at the time of the call: a batch is a few waves of resident blocks, and the draining
  // tail of one launch + the launch gap overlap the next launch instead. With GALE_STREAM_ORDERED the
  // kernels run on the caller's stream itself.
  static constexpr int kLaunchStreams = 2;
  cudaStream_t launch[kLaunchStreams] = {nullptr, nullptr};
  int32_t* h_err = nullptr;  // mapped pinned; the kernels write guard codes here
  std::atomic<long long> submitted{0}, popped{0};
  size_t workspace_used = 0, index_bytes = 0;
  double create_ms = 0;
  float tune_ms[2] = {0.f, 0.f};  // sample-batch time of the dense / walk kernel at create (0 = not timed)
};

namespace {
void free_mesh(gale_mesh* m) {  // also the error path of create: releases whatever exists so far
  if (!m) return;
  if (m->side) { cudaStreamSynchronize(m->side); cudaStreamDestroy(m->side); }
  for (cudaStream_t& ls : m->launch)
    if (ls) { cudaStreamSynchronize(ls); cudaStreamDestroy(ls); ls = nullptr; }
  for (auto& s : m->slots) {
    if (s->pinned) cudaFreeHost(s->pinned);
    if (s->ev_submit) cudaEventDestroy(s->ev_submit);
    if (s->ev_start) cudaEventDestroy(s->ev_start);
    if (s->ev_done) cudaEventDestroy(s->ev_done);
    if (s->ev_ready) cudaEventDestroy(s->ev_ready);
  }
  if (m->h_err) cudaFreeHost(m->h_err);
  cudaGetLastError();
  delete m;
}

int build_mesh(std::unique_ptr<Plan> p, void* d_workspace, size_t workspace_bytes, cudaStream_t st, gale_mesh_t** out) {
  if (!d_workspace || reinterpret_cast<uintptr_t>(d_workspace) % kAlign) return GALE_ERR_WORKSPACE;
  if (total_workspace(*p) > workspace_bytes) return GALE_ERR_WORKSPACE;
  const auto t0 = std::chrono::steady_clock::now();
  gale_mesh* m = new gale_mesh();
  struct Guard { gale_mesh* m; ~Guard() { free_mesh(m); } } guard{m};
  m->dim = p->dim; m->D = p->dim + 1; m->maxB = p->maxB; m->queue_depth = p->queue_depth;
  m->stream_ordered = (p->flags & GALE_STREAM_ORDERED) != 0;
  char* base = static_cast<char*>(d_workspace);
  const IndexLayout IL = index_layout(*p);
  auto put = [&](size_t at, const void* src, size_t bytes) -> int {
    if (bytes) GALE_CUDA(cudaMemcpyAsync(base + at, src, bytes, cudaMemcpyHostToDevice, st));
    return GALE_OK;
  };
  int rc;
  if ((rc = put(IL.first_tet, p->first_tet.data(), p->first_tet.size() * 4)) ||
      (rc = put(IL.opp_first, p->opp_first.data(), p->opp_first.size() * 4)) ||
      (rc = put(IL.opp_perm, p->opp_perm.data(), p->opp_perm.size() * 4)) ||
      (rc = put(IL.cl_tile_begin, p->cl_tile_begin.data(), p->cl_tile_begin.size() * 4)) ||
      (rc = put(IL.tiles, p->tiles.data(), p->tiles.size() * sizeof(TileDesc))) ||
      (rc = put(IL.tex, p->tex.data(), p->tex.size() * 4)) || (rc = put(IL.gid, p->gid.data(), p->gid.size() * 4)) ||
      (rc = p->cfg.lb == 1 ? put(IL.loc, p->loc8.data(), p->loc8.size()) : put(IL.loc, p->loc.data(), p->loc.size() * 2)))
    return rc;
  m->dm.T = p->dT;
  m->dm.first_tet = reinterpret_cast<int32_t*>(base + IL.first_tet);
  m->dm.opp_first = reinterpret_cast<int32_t*>(base + IL.opp_first);
  m->dm.opp_perm = reinterpret_cast<int32_t*>(base + IL.opp_perm);
  m->dm.cluster_tile_begin = reinterpret_cast<int32_t*>(base + IL.cl_tile_begin);
  m->dm.tiles = reinterpret_cast<TileDesc*>(base + IL.tiles);
  m->dm.tex = reinterpret_cast<int32_t*>(base + IL.tex);
  m->dm.gid = reinterpret_cast<int32_t*>(base + IL.gid);
  m->dm.loc = base + IL.loc;
  m->index_bytes = IL.total;
  // the index tables can be dropped on the host once uploaded (keep the small per-cluster ones)
  GALE_CUDA(cudaStreamSynchronize(st));
  std::vector<int32_t>().swap(p->opp_perm);
  std::vector<int32_t>().swap(p->tex);
  std::vector<int32_t>().swap(p->gid);
  std::vector<uint16_t>().swap(p->loc);
  std::vector<uint8_t>().swap(p->loc8);
  std::vector<int32_t>().swap(p->opp_first);

  GALE_CUDA(cudaHostAlloc(reinterpret_cast<void**>(&m->h_err), 64, cudaHostAllocMapped));
  *m->h_err = 0;
  GALE_CUDA(cudaHostGetDevicePointer(reinterpret_cast<void**>(&m->dm.err), m->h_err, 0));

  m->cap = slot_capacity_layout(*p, m->maxB);
  const int nslots = slots_of(p->queue_depth, p->device_ring);
  size_t o = IL.total;
  for (int i = 0; i < nslots; ++i) {
    auto s = std::make_unique<Slot>();
    s->dev = base + o;
    o += m->cap.total;
    Slot* sp = s.get();
    m->slots.push_back(std::move(s));  // owned by the handle from here on (error paths free it)
    if (p->queue_depth > 0) GALE_CUDA(cudaHostAlloc(reinterpret_cast<void**>(&sp->pinned), std::max<size_t>(m->cap.total, 16), cudaHostAllocDefault));
    GALE_CUDA(cudaEventCreateWithFlags(&sp->ev_submit, cudaEventDisableTiming));
    GALE_CUDA(cudaEventCreate(&sp->ev_start));
    GALE_CUDA(cudaEventCreate(&sp->ev_done));
    GALE_CUDA(cudaEventCreate(&sp->ev_ready));
  }
  if (o > workspace_bytes) return GALE_ERR_WORKSPACE;  // cannot happen: total_workspace() uses the same layout
  m->workspace_used = o;
  if (p->queue_depth > 0) GALE_CUDA(cudaStreamCreateWithFlags(&m->side, cudaStreamNonBlocking));
  if (!m->stream_ordered)
    for (int i = 0; i < gale_mesh::kLaunchStreams; ++i) GALE_CUDA(cudaStreamCreateWithFlags(&m->launch[i], cudaStreamNonBlocking));
  GALE_CUDA(allow_max_smem(kernel_for(m->D, p->NT, false, p->cfg.lb)));
  if (p->walk_ok) GALE_CUDA(cudaFuncSetAttribute(walk_kernel_for(m->D, p->w_NT, p->cfg.lb), cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit));
  const uint32_t force = p->flags & (GALE_KERNEL_DENSE | GALE_KERNEL_WALK);
  const bool may_walk = p->walk_ok;
  m->plan = std::move(p);
  if (force == GALE_KERNEL_WALK && !may_walk) { g_last_error = "the walk kernel cannot run these tiles (capacity limits)"; return GALE_ERR_UNSUPPORTED; }
  m->kernel = force == GALE_KERNEL_WALK ? 1 : 0;
  if (force == 0 && may_walk && m->plan->nC > 0 && m->plan->nT > 0) {
    // Pick the kernel by measurement: one sample batch (the middle clusters) through each, best of 3
    // event-timed runs after 1 warm-up. Uniform vertex stars favour the walk kernel, irregular ones the dense.
    const int nC = m->plan->nC, n = std::min(m->maxB, nC);
    std::vector<int32_t> ids(static_cast<size_t>(n), 0);
    for (int i = 0; i < n; ++i) ids[size_t(i)] = (nC - n) / 2 + i;
    float best[2] = {1e30f, 1e30f};
    for (int k = 0; k < 2; ++k) {
      m->kernel = k;
      for (int rep = 0; rep < 4; ++rep) {
        int rc2 = gale_cluster_batch_compute(m, GALE_REL_ALL, ids.data(), n, st);
        gale_batch_view_t v;
        if (rc2 == GALE_OK) rc2 = gale_queue_pop(m, &v, -1);
        if (rc2 != GALE_OK) return rc2;
        if (rep > 0) best[k] = std::min(best[k], v.kernel_ms);
        if ((rc2 = gale_queue_release(m, &v)) != GALE_OK) return rc2;
      }
    }
    m->kernel = best[1] < best[0] ? 1 : 0;
    m->tune_ms[0] = best[0]; m->tune_ms[1] = best[1];
    m->submitted.store(0); m->popped.store(0);  // the sample batches are not the caller's: sequence numbers restart
  }
  m->create_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count() + m->plan->analyse_ms;
  guard.m = nullptr;
  *out = m;
  return GALE_OK;
}
}  // namespace

extern "C" {

const char* gale_status_string(int32_t s) {
  switch (s) {
    case GALE_OK: return "GALE_OK";
    case GALE_ERR_INVALID_ARG: return "GALE_ERR_INVALID_ARG";
    case GALE_ERR_NOT_CANONICAL: return "GALE_ERR_NOT_CANONICAL";
    case GALE_ERR_DEGENERATE: return "GALE_ERR_DEGENERATE";
    case GALE_ERR_NONMANIFOLD: return "GALE_ERR_NONMANIFOLD";
    case GALE_ERR_BAD_CLUSTER: return "GALE_ERR_BAD_CLUSTER";
    case GALE_ERR_WOULD_BLOCK: return "GALE_ERR_WOULD_BLOCK";
    case GALE_ERR_EMPTY: return "GALE_ERR_EMPTY";
    case GALE_ERR_WORKSPACE: return "GALE_ERR_WORKSPACE";
    case GALE_ERR_CUDA: return "GALE_ERR_CUDA";
    case GALE_ERR_UNSUPPORTED: return "GALE_ERR_UNSUPPORTED";
    default: return "GALE_ERR_UNKNOWN";
  }
}
const char* gale_last_error(void) { return g_last_error.c_str(); }

int32_t gale_plan_create(const gale_mesh_desc_t* desc, void* cuda_stream, gale_plan_t** out) {
  if (!out) return GALE_ERR_INVALID_ARG;
  int rc = check_desc(desc);
  if (rc != GALE_OK) return rc;
  if ((rc = check_device()) != GALE_OK) return rc;
  std::unique_ptr<Plan> p;
  if ((rc = analyse(*desc, static_cast<cudaStream_t>(cuda_stream), p)) != GALE_OK) return rc;
  *out = new gale_plan{std::move(p)};
  return GALE_OK;
}

int32_t gale_plan_workspace_bytes(const gale_plan_t* plan, size_t* out_bytes) {
  if (!plan || !plan->plan || !out_bytes) return GALE_ERR_INVALID_ARG;
  *out_bytes = total_workspace(*plan->plan);
  return GALE_OK;
}

int32_t gale_plan_destroy(gale_plan_t* plan) {
  if (!plan) return GALE_ERR_INVALID_ARG;
  delete plan;
  return GALE_OK;
}

int32_t gale_mesh_create_planned(gale_plan_t* plan, void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                                 gale_mesh_t** out) {
  if (!plan || !plan->plan || !out) return GALE_ERR_INVALID_ARG;
  return build_mesh(std::move(plan->plan), d_workspace, workspace_bytes, static_cast<cudaStream_t>(cuda_stream), out);
}

int32_t gale_mesh_workspace_bytes(const gale_mesh_desc_t* desc, void* cuda_stream, size_t* out_bytes) {
  if (!out_bytes) return GALE_ERR_INVALID_ARG;
  gale_plan_t* plan = nullptr;
  int rc = gale_plan_create(desc, cuda_stream, &plan);
  if (rc != GALE_OK) return rc;
  *out_bytes = total_workspace(*plan->plan);
  delete plan;
  return GALE_OK;
}

int32_t gale_mesh_create(const gale_mesh_desc_t* desc, void* cuda_stream, gale_mesh_t** out) {
  if (!out) return GALE_ERR_INVALID_ARG;
  int rc = check_desc(desc);
  if (rc != GALE_OK) return rc;
  if (!desc->d_workspace || reinterpret_cast<uintptr_t>(desc->d_workspace) % kAlign) return GALE_ERR_WORKSPACE;
  gale_plan_t* plan = nullptr;
  if ((rc = gale_plan_create(desc, cuda_stream, &plan)) != GALE_OK) return rc;
  rc = build_mesh(std::move(plan->plan), desc->d_workspace, desc->workspace_bytes, static_cast<cudaStream_t>(cuda_stream), out);
  delete plan;
  return rc;
}

int32_t gale_mesh_info(const gale_mesh_t* m, gale_mesh_info_t* out) {
  if (!m || !out) return GALE_ERR_INVALID_ARG;
  const Plan& p = *m->plan;
  out->tile_vertices = p.tv;
  out->num_tiles = p.nTiles;
  out->num_external_refs = p.ext_refs;
  out->vt_nnz = p.vt_total;
  out->vv_nnz = p.vv_total;
  out->smem_bytes = m->kernel == 1 ? p.w_smem : p.smem_bytes;
  out->max_staged = p.cfg.smax;
  out->slot_bytes = m->cap.total;
  out->workspace_used = m->workspace_used;
  out->create_ms = m->create_ms;
  out->local_id_bytes = p.cfg.lb;
  out->block_threads = m->kernel == 1 ? p.w_NT : p.NT;
  out->index_bytes = m->index_bytes;
  out->kernel_variant = m->kernel;
  out->tune_dense_ms = m->tune_ms[0];
  out->tune_walk_ms = m->tune_ms[1];
  out->reserved = 0;
  return GALE_OK;
}

int32_t gale_cluster_batch_compute(gale_mesh_t* m, uint32_t relation_mask, const int32_t* h_cluster_ids,
                                   int32_t n_clusters, void* cuda_stream) {
  if (!m || (relation_mask & ~uint32_t(GALE_REL_ALL)) || relation_mask == 0 || n_clusters < 0 ||
      (n_clusters > 0 && !h_cluster_ids))
    return GALE_ERR_INVALID_ARG;
  if (n_clusters > m->maxB) return GALE_ERR_BAD_CLUSTER;
  const Plan& p = *m->plan;
  for (int i = 0; i < n_clusters; ++i)
    if (h_cluster_ids[i] < 0 || h_cluster_ids[i] >= p.nC) return GALE_ERR_BAD_CLUSTER;
  const long long seq = m->submitted.load();
  Slot& s = *m->slots[size_t(seq % (long long)m->slots.size())];
  if (s.state.load(std::memory_order_acquire) != SLOT_FREE) return GALE_ERR_WOULD_BLOCK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int D = m->D;
  const auto t_prep = std::chrono::steady_clock::now();

  // batch set-up (a0): row / nnz bases of every requested cluster, in request order
  s.seq = seq; s.n = n_clusters; s.mask = relation_mask;
  s.ids.assign(h_cluster_ids, h_cluster_ids + n_clusters);
  s.row_begin.assign(n_clusters + 1, 0);
  s.tt_row_begin.assign(n_clusters + 1, 0);
  std::vector<long long> vtb(n_clusters + 1, 0), vvb(n_clusters + 1, 0);
  for (int i = 0; i < n_clusters; ++i) {
    const int c = s.ids[i];
    const long long rows = p.cl_off[c + 1] - p.cl_off[c];
    const long long ttr = p.cl_t_lo[c + 1] - p.cl_t_lo[c];
    if (s.row_begin[i] + rows >= (1LL << 31) - 1 || vtb[i] + p.cl_vt[c] >= (1LL << 31) - 1 ||
        (s.tt_row_begin[i] + ttr) * D >= (1LL << 31) - 1)
      return GALE_ERR_INVALID_ARG;
    s.row_begin[i + 1] = int32_t(s.row_begin[i] + rows);
    s.tt_row_begin[i + 1] = int32_t(s.tt_row_begin[i] + ttr);
    vtb[i + 1] = vtb[i] + p.cl_vt[c];
    vvb[i + 1] = vvb[i] + p.cl_vv[c];
  }
  s.rows = s.row_begin[n_clusters]; s.vt_nnz = vtb[n_clusters]; s.vv_nnz = vvb[n_clusters];
  s.tt_rows = s.tt_row_begin[n_clusters];
  // compact section layout of this batch (one D2H copy of `used.total` bytes)
  {
    size_t o = 0;
    s.used.vt_off = o; if (relation_mask & GALE_REL_VT) o = up(o + size_t(s.rows + 1) * 4, 16);
    s.used.vt_idx = o; if (relation_mask & GALE_REL_VT) o = up(o + size_t(s.vt_nnz) * 4, 16);
    s.used.vv_off = o; if (relation_mask & GALE_REL_VV) o = up(o + size_t(s.rows + 1) * 4, 16);
    s.used.vv_idx = o; if (relation_mask & GALE_REL_VV) o = up(o + size_t(s.vv_nnz) * 4, 16);
    s.used.tt = o;     if (relation_mask & GALE_REL_TT) o = up(o + size_t(s.tt_rows) * D * 4, 16);
    s.used.total = o;
    if (o > m->cap.total) return GALE_ERR_WORKSPACE;
  }
  gale::OutPtrs O{};
  O.vt_offsets = reinterpret_cast<int32_t*>(s.dev + s.used.vt_off);
  O.vt_indices = reinterpret_cast<int32_t*>(s.dev + s.used.vt_idx);
  O.vv_offsets = reinterpret_cast<int32_t*>(s.dev + s.used.vv_off);
  O.vv_indices = reinterpret_cast<int32_t*>(s.dev + s.used.vv_idx);
  O.tt_indices = reinterpret_cast<int32_t*>(s.dev + s.used.tt);

  const bool walk = m->kernel == 1;
  SmemCfg cfg = walk ? walk_cfg_for_mask(p.cfg, relation_mask) : cfg_for_mask(p.cfg, relation_mask, false);
  const gale::SmemLayout lay = layout_for(D, cfg);
  const gale::WalkLayout wlay = walk_layout_for(D, cfg);
#if GALE_CHECK_BOUNDS
  // negative control of the bounds-checked build: understate one capacity (the layout keeps its real
  // size) so that the kernel's checks must fire
  if (std::getenv("GALE_CHECK_SELFTEST") && cfg.vt_max > 8) cfg.vt_max -= 8;
#endif
  const int smem = walk ? wlay.total : lay.total;
  // everything the caller enqueued on its stream so far (e.g. the upload of the simplices) comes first
  cudaStream_t run = m->stream_ordered ? st : m->launch[seq % gale_mesh::kLaunchStreams];
  if (!m->stream_ordered) {
    GALE_CUDA(cudaEventRecord(s.ev_submit, st));
    GALE_CUDA(cudaStreamWaitEvent(run, s.ev_submit, 0));
  }
  GALE_CUDA(cudaEventRecord(s.ev_start, run));
  for (int b = 0; b < std::max(1, n_clusters); b += gale::kMaxBatch) {
    gale::BatchParams P{};
    const int nb = std::max(0, std::min(gale::kMaxBatch, n_clusters - b));
    P.n_clusters = nb; P.mask = relation_mask;
    P.total_rows = int(s.rows); P.total_vt_nnz = int(s.vt_nnz); P.total_vv_nnz = int(s.vv_nnz);
    for (int i = 0; i < nb; ++i) {
      const int c = s.ids[b + i];
      P.tile_prefix[i + 1] = P.tile_prefix[i] + (p.cl_tile_begin[c + 1] - p.cl_tile_begin[c]);
      P.cluster[i] = c;
      P.row_base[i] = s.row_begin[b + i];
      P.vt_base[i] = int(vtb[b + i]);
      P.vv_base[i] = int(vvb[b + i]);
      P.tt_base[i] = s.tt_row_begin[b + i];
    }
    {  // all clusters with the same tile count: the kernel divides instead of searching tile_prefix
      const int per = nb > 0 ? P.tile_prefix[1] : 0;
      bool uniform = per > 0;
      for (int i = 0; i < nb && uniform; ++i) uniform = P.tile_prefix[i + 1] - P.tile_prefix[i] == per;
      P.uniform_tiles = uniform ? per : 0;
    }
    const int grid = std::max(1, P.tile_prefix[nb]);
    if (walk) walk_kernel_for(D, p.w_NT, p.cfg.lb)<<<grid, p.w_NT, smem, run>>>(m->dm, P, cfg, wlay, O);
    else kernel_for(D, p.NT, false, p.cfg.lb)<<<grid, p.NT, smem, run>>>(m->dm, P, cfg, lay, O);
    GALE_CUDA(cudaGetLastError());
  }
  GALE_CUDA(cudaEventRecord(s.ev_done, run));
  if (m->queue_depth > 0) {  // a7: D2H into the pinned slot on the side stream
    GALE_CUDA(cudaStreamWaitEvent(m->side, s.ev_done, 0));
    if (s.used.total) GALE_CUDA(cudaMemcpyAsync(s.pinned, s.dev, s.used.total, cudaMemcpyDeviceToHost, m->side));
    GALE_CUDA(cudaEventRecord(s.ev_ready, m->side));
  }
  s.t_submit = std::chrono::steady_clock::now();
  s.prep_ms = std::chrono::duration<float, std::milli>(s.t_submit - t_prep).count();
  s.state.store(SLOT_SUBMITTED, std::memory_order_release);
  m->submitted.store(seq + 1);
  return GALE_OK;
}

int32_t gale_queue_pop(gale_mesh_t* m, gale_batch_view_t* out, int32_t timeout_ms) {
  if (!m || !out) return GALE_ERR_INVALID_ARG;
  const long long seq = m->popped.load();
  if (seq >= m->submitted.load()) return GALE_ERR_EMPTY;
  Slot& s = *m->slots[size_t(seq % (long long)m->slots.size())];
  if (s.state.load(std::memory_order_acquire) != SLOT_SUBMITTED) return GALE_ERR_EMPTY;
  cudaEvent_t ev = m->queue_depth > 0 ? s.ev_ready : s.ev_done;
  if (timeout_ms < 0) {
    GALE_CUDA(cudaEventSynchronize(ev));
  } else {
    const auto deadline = std::chrono::steady_clock::now() + std::chrono::milliseconds(timeout_ms);
    for (;;) {
      cudaError_t q = cudaEventQuery(ev);
      if (q == cudaSuccess) break;
      if (q != cudaErrorNotReady) { g_last_error = cudaGetErrorString(q); return GALE_ERR_CUDA; }
      if (std::chrono::steady_clock::now() >= deadline) return GALE_ERR_WOULD_BLOCK;
      std::this_thread::yield();
    }
  }
  if (*static_cast<volatile int32_t*>(m->h_err) != 0) {
    g_last_error = "device capacity guard fired: code " + std::to_string(*m->h_err);
    return GALE_ERR_WORKSPACE;
  }
  const char* b = m->queue_depth > 0 ? s.pinned : s.dev;
  std::memset(out, 0, sizeof(*out));
  out->sequence = s.seq; out->n_clusters = s.n; out->relation_mask = s.mask; out->dim = m->dim;
  out->on_device = m->queue_depth > 0 ? 0 : 1;
  out->cluster_ids = s.ids.data();
  out->vt_row_begin = s.row_begin.data();
  out->tt_row_begin = s.tt_row_begin.data();
  if (s.mask & GALE_REL_VT) {
    out->vt_rows = s.rows; out->vt_nnz = s.vt_nnz;
    out->vt_offsets = reinterpret_cast<const int32_t*>(b + s.used.vt_off);
    out->vt_indices = reinterpret_cast<const int32_t*>(b + s.used.vt_idx);
  }
  if (s.mask & GALE_REL_VV) {
    out->vv_rows = s.rows; out->vv_nnz = s.vv_nnz;
    out->vv_offsets = reinterpret_cast<const int32_t*>(b + s.used.vv_off);
    out->vv_indices = reinterpret_cast<const int32_t*>(b + s.used.vv_idx);
  }
  if (s.mask & GALE_REL_TT) {
    out->tt_rows = s.tt_rows;
    out->tt_indices = reinterpret_cast<const int32_t*>(b + s.used.tt);
  }
  float ms = 0.f;
  if (cudaEventElapsedTime(&ms, s.ev_start, s.ev_done) != cudaSuccess) { cudaGetLastError(); ms = 0.f; }
  out->kernel_ms = ms;
  ms = 0.f;
  if (m->queue_depth > 0 && cudaEventElapsedTime(&ms, s.ev_done, s.ev_ready) != cudaSuccess) { cudaGetLastError(); ms = 0.f; }
  out->d2h_ms = ms;  // includes the time the copy waited for earlier copies on the side stream
  out->prep_ms = s.prep_ms;
  out->queue_ms = std::chrono::duration<float, std::milli>(std::chrono::steady_clock::now() - s.t_submit).count();
  out->slot = int32_t(seq % (long long)m->slots.size());
  s.state.store(SLOT_POPPED, std::memory_order_release);
  m->popped.store(seq + 1);
  return GALE_OK;
}

int32_t gale_queue_release(gale_mesh_t* m, const gale_batch_view_t* view) {
  if (!m || !view || view->slot < 0 || view->slot >= int(m->slots.size())) return GALE_ERR_INVALID_ARG;
  Slot& s = *m->slots[size_t(view->slot)];
  if (s.state.load(std::memory_order_acquire) != SLOT_POPPED || s.seq != view->sequence) return GALE_ERR_INVALID_ARG;
  s.state.store(SLOT_FREE, std::memory_order_release);
  return GALE_OK;
}

int32_t gale_destroy(gale_mesh_t* m) {
  if (!m) return GALE_ERR_INVALID_ARG;
  for (auto& s : m->slots) {
    if (s->ev_done) cudaEventSynchronize(s->ev_done);
    if (m->queue_depth > 0 && s->ev_ready && s->state.load() != SLOT_FREE) cudaEventSynchronize(s->ev_ready);
  }
  free_mesh(m);
  return GALE_OK;
}

}  // extern "C"
