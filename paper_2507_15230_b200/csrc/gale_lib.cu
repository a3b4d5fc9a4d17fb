// gale_lib.cu — C-ABI boundary of the GALE relation hot path (include/gale.h).
//
// Host side of the paper's producer: initialization (I_T, T_ex, interval arrays),
// the leader producer's batch set-up and launch and the bounded queue of
// pre-allocated result buffers handed to consumers. Every relation entry is
// computed by the kernels in gale_kernels.cuh; nothing here computes VT/VV/TT on the CPU.
#include "gale_kernels.cuh"
#include "gale_walk.cuh"
#include "gale_init.cuh"
#include "gale_sub.cuh"
#include "gale_canon.cuh"

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

// Device memory owned by the library for the duration of the initialization.
struct DevMem {
  void* p = nullptr;
  size_t bytes = 0;
  DevMem() = default;
  DevMem(const DevMem&) = delete;
  DevMem& operator=(const DevMem&) = delete;
  ~DevMem() { release(); }
  void release() { if (p) cudaFree(p); p = nullptr; bytes = 0; }
  int alloc(size_t n) {
    release();
    bytes = n;
    GALE_CUDA(cudaMalloc(&p, std::max<size_t>(n, 256)));
    return GALE_OK;
  }
  template <class T> T* as() const { return static_cast<T*>(p); }
};

// ---- result of the initialization analysis -----------------------------------------
struct Plan {
  // key
  const int32_t* dT = nullptr;
  int dim = 0, nV = 0, nC = 0, tv_req = 0, maxB = 1, queue_depth = 0, device_ring = 0;
  long long nT = 0;
  uint32_t flags = 0;
  std::vector<int32_t> cl_off;
  // the index, built on the device (gale_init.cuh); owned here until build_mesh copies it into the
  // caller's workspace
  int tv = 0, nTiles = 0, NT = 0;
  DevMem d_first_tet, d_opp_first, d_opp_perm, d_tex, d_gid, d_loc;
  size_t n_tex = 0, n_gid = 0, loc_bytes = 0;   // element counts / bytes of tex, gid, loc incl. padding
  std::vector<int32_t> cl_tile_begin;
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
  size_t vt_off = 0, vt_idx = 0, vv_off = 0, vv_idx = 0, tt = 0, ve_idx = 0, vf_off = 0, vf_idx = 0;
  size_t cob_off[3] = {0, 0, 0}, cob_idx[3] = {0, 0, 0};  // ET, FT, EF (gale::sub::COB_*)
  size_t total = 0;
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
  if (p.flags & GALE_WITH_EDGES) { L.ve_idx = o; o = up(o + size_t(maxB) * p.max_vv * 4); }
  if (p.flags & GALE_WITH_FACETS) {  // |VF(v)| <= 3 |VT(v)|: every triangle at v lies in a simplex of its star
    L.vf_off = o; o = up(o + (size_t(maxB) * p.max_rows + 1) * 4);
    L.vf_idx = o; o = up(o + size_t(maxB) * p.max_vt * 3 * 4);
  }
  if (p.flags & GALE_WITH_COBOUNDARY) {
    // bounds known before E / F exist: an edge / triangle internal to a cluster has its lowest vertex a there and
    // lies in a simplex of VT(a); a simplex has 3 edges and 3 triangles with a given lowest vertex
    const size_t rows[3] = {size_t(p.max_vv), size_t(p.max_vt) * 3, size_t(p.max_vv)};
    const size_t nnz[3] = {size_t(p.max_vt) * 3, size_t(p.max_vt) * 3, size_t(p.max_vt) * 6};
    for (int k = 0; k < 3; ++k) {
      L.cob_off[k] = o; o = up(o + (size_t(maxB) * rows[k] + 1) * 4);
      L.cob_idx[k] = o; o = up(o + size_t(maxB) * nnz[k] * 4);
    }
  }
  L.total = o;
  return L;
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

inline int threads_for_tile(int tv) { return tv > 128 ? 256 : 128; }  // NT >= tv (one thread per row in P2); 256 threads for 32-vertex tiles measured -25 %

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
template <int D, int LB, bool ALL>
WalkFn walk_for_nt(int NT) {
  return NT == 512 ? gale::gale_walk_kernel<D, 512, LB, ALL>
                   : (NT == 256 ? gale::gale_walk_kernel<D, 256, LB, ALL>
                                : (NT == 128 ? gale::gale_walk_kernel<D, 128, LB, ALL> : gale::gale_walk_kernel<D, 64, LB, ALL>));
}
template <bool ALL>
WalkFn walk_kernel_for_all(int D, int NT, int lb) {
  if (D == 4) return lb == 1 ? walk_for_nt<4, 1, ALL>(NT) : walk_for_nt<4, 2, ALL>(NT);
  return lb == 1 ? walk_for_nt<3, 1, ALL>(NT) : walk_for_nt<3, 2, ALL>(NT);
}
WalkFn walk_kernel_for(int D, int NT, int lb, bool all = false) {
  return all ? walk_kernel_for_all<true>(D, NT, lb) : walk_kernel_for_all<false>(D, NT, lb);
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

// Host <-> device helpers of the initialization.
template <class V>
int upload_vec(DevMem& d, const V& v, cudaStream_t st) {
  int rc = d.alloc(v.size() * sizeof(typename V::value_type));
  if (rc != GALE_OK) return rc;
  if (!v.empty()) GALE_CUDA(cudaMemcpyAsync(d.p, v.data(), v.size() * sizeof(typename V::value_type), cudaMemcpyHostToDevice, st));
  return GALE_OK;
}
template <class T>
int download_vec(std::vector<T>& v, const void* d, size_t n, cudaStream_t st) {
  v.resize(n);
  if (n) GALE_CUDA(cudaMemcpyAsync(v.data(), d, n * sizeof(T), cudaMemcpyDeviceToHost, st));
  GALE_CUDA(cudaStreamSynchronize(st));
  return GALE_OK;
}
inline int blocks_for(long long n, int threads) { return int(std::max<long long>(1, (n + threads - 1) / threads)); }

constexpr int kRefCap = 16384;  // vertex references (D * staged simplices) a tile may have in the halo pass

// Tiles of `tv` vertices on the device: T_ex lists, halo vertices, the tile-local encoding
// of the staged simplices. The host sees per-tile scalars only. fits = false: a tile exceeds a kernel
// limit at this tile size (the caller retries with a smaller one).
template <int D>
int build_tiles_device(Plan& p, int tv, cudaStream_t st, bool& fits) {
  namespace gi = gale::init;
  fits = true;
  p.tv = tv;
  p.NT = threads_for_tile(tv);
  // tile table (host: one entry per tile)
  std::vector<int32_t> vlo, nrows, tile_cluster;
  p.cl_tile_begin.assign(p.nC + 1, 0);
  for (int c = 0; c < p.nC; ++c) {
    p.cl_tile_begin[c] = int(vlo.size());
    for (int v = p.cl_off[c]; v < p.cl_off[c + 1]; v += tv) {
      vlo.push_back(v);
      nrows.push_back(std::min(tv, p.cl_off[c + 1] - v));
      tile_cluster.push_back(c);
    }
  }
  const int nTiles = int(vlo.size());
  p.cl_tile_begin[p.nC] = nTiles;
  p.nTiles = nTiles;
  p.tiles.assign(nTiles, TileDesc{});
  p.ext_refs = 0; p.staged_padded = 0; p.n_tex = 4; p.n_gid = 4; p.loc_bytes = 64;
  p.cfg = SmemCfg{};
  p.cfg.tv = tv; p.cfg.smax = 4; p.cfg.sext = 4; p.cfg.sint = 2; p.cfg.nloc = 4; p.cfg.lb = 1;
  p.cfg.WT = 1; p.cfg.WV = 1;
  int rc;
  if (nTiles == 0) {
    if ((rc = p.d_tex.alloc(16)) || (rc = p.d_gid.alloc(16)) || (rc = p.d_loc.alloc(64))) return rc;
    return GALE_OK;
  }
  const int TB = 256;
  DevMem d_vlo, d_nrows, d_tile_of, d_tlo, d_sint, d_cnt, d_scan, d_raw, d_cursor;
  if ((rc = upload_vec(d_vlo, vlo, st)) || (rc = upload_vec(d_nrows, nrows, st)) ||
      (rc = d_tile_of.alloc(size_t(std::max(p.nV, 1)) * 4)) || (rc = d_tlo.alloc(size_t(nTiles) * 4)) ||
      (rc = d_sint.alloc(size_t(nTiles) * 4)) || (rc = d_cnt.alloc(size_t(nTiles + 1) * 4)) ||
      (rc = d_scan.alloc((size_t(nTiles) / gi::kScanChunk + 2) * 4)))
    return rc;
  gi::k_tile_of<<<blocks_for(nTiles, TB), TB, 0, st>>>(d_vlo.as<int32_t>(), d_nrows.as<int32_t>(), nTiles, d_tile_of.as<int32_t>());
  gi::k_tile_internal<<<blocks_for(nTiles, TB), TB, 0, st>>>(p.d_first_tet.as<int32_t>(), d_vlo.as<int32_t>(), d_nrows.as<int32_t>(),
                                                             nTiles, d_tlo.as<int32_t>(), d_sint.as<int32_t>());
  GALE_CUDA(cudaMemsetAsync(d_cnt.p, 0, size_t(nTiles + 1) * 4, st));
  if (p.nT) gi::k_external<D, true><<<blocks_for(p.nT, TB), TB, 0, st>>>(p.dT, p.nT, d_tile_of.as<int32_t>(), d_cnt.as<int32_t>(), nullptr);
  GALE_CUDA(gi::exclusive_scan_i32(d_cnt.as<int32_t>(), nTiles + 1, d_scan.as<int32_t>(), st));  // -> raw_off
  std::vector<int32_t> raw_off, t_lo, s_int;
  if ((rc = download_vec(raw_off, d_cnt.p, size_t(nTiles) + 1, st)) || (rc = download_vec(t_lo, d_tlo.p, size_t(nTiles), st)) ||
      (rc = download_vec(s_int, d_sint.p, size_t(nTiles), st)))
    return rc;
  p.ext_refs = raw_off[nTiles];
  // per-tile scalars, padded offsets, limits that need no halo
  std::vector<int32_t> s_ext(nTiles);
  std::vector<long long> stg_off(nTiles), tex_off(nTiles);
  long long stg = 0, texo = 0, smax = 4, sextm = 4, sintm = 2;
  for (int i = 0; i < nTiles; ++i) {
    TileDesc& d = p.tiles[i];
    const int c = tile_cluster[i];
    d.v_lo = vlo[i]; d.nrows = nrows[i];
    d.t_lo = t_lo[i]; d.s_int = s_int[i];
    d.s_ext = s_ext[i] = raw_off[i + 1] - raw_off[i];
    d.row_rel = d.v_lo - p.cl_off[c];
    d.c_rows = p.cl_off[c + 1] - p.cl_off[c];
    d.tt_rel = d.t_lo - p.cl_t_lo[c];
    d.stg_off = stg_off[i] = stg;
    d.tex_off = tex_off[i] = texo;
    const long long S = (long long)d.s_int + d.s_ext;
    if (S > (D == 4 ? gale::kMaxStaged4 : gale::kMaxStaged3) || S * D > kRefCap) { fits = false; return GALE_OK; }
    stg += pad_to(S, 4);
    texo += pad_to(d.s_ext, 4);
    smax = std::max(smax, pad_to(S, 4));
    sextm = std::max(sextm, pad_to(d.s_ext, 4));
    sintm = std::max(sintm, pad_to(d.s_int, 2));
  }
  p.staged_padded = stg;
  p.n_tex = size_t(texo) + 4;
  // T_ex lists: scatter, then sort each tile's list ascending into its padded place
  DevMem d_texoff, d_stgoff, d_sext;
  if ((rc = d_raw.alloc(size_t(std::max<long long>(p.ext_refs, 1)) * 4)) || (rc = d_cursor.alloc(size_t(nTiles + 1) * 4)) ||
      (rc = p.d_tex.alloc(p.n_tex * 4)) || (rc = upload_vec(d_texoff, tex_off, st)) || (rc = upload_vec(d_stgoff, stg_off, st)) ||
      (rc = upload_vec(d_sext, s_ext, st)))
    return rc;
  GALE_CUDA(cudaMemcpyAsync(d_cursor.p, d_cnt.p, size_t(nTiles + 1) * 4, cudaMemcpyDeviceToDevice, st));
  if (p.nT) gi::k_external<D, false><<<blocks_for(p.nT, TB), TB, 0, st>>>(p.dT, p.nT, d_tile_of.as<int32_t>(), d_cursor.as<int32_t>(), d_raw.as<int32_t>());
  {
    const int smem = gi::pow2_ceil(int(sextm)) * 4;
    GALE_CUDA(cudaFuncSetAttribute(gi::k_sort_external, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit - 2048));
    gi::k_sort_external<<<nTiles, TB, smem, st>>>(d_raw.as<int32_t>(), d_cnt.as<int32_t>(), d_texoff.as<long long>(), p.d_tex.as<int32_t>());
    GALE_CUDA(cudaGetLastError());
  }
  d_raw.release(); d_cursor.release(); d_tile_of.release();
  // halo of every tile: count, then (offsets known) write gid and loc
  DevMem d_nlo, d_nhalo, d_gidoff, d_flag;
  if ((rc = d_nlo.alloc(size_t(nTiles) * 4)) || (rc = d_nhalo.alloc(size_t(nTiles) * 4)) || (rc = d_flag.alloc(4))) return rc;
  GALE_CUDA(cudaMemsetAsync(d_flag.p, 0, 4, st));
  gi::TileArrays A{};
  A.vlo = d_vlo.as<int32_t>(); A.nrows = d_nrows.as<int32_t>(); A.t_lo = d_tlo.as<int32_t>(); A.s_int = d_sint.as<int32_t>();
  A.s_ext = d_sext.as<int32_t>(); A.tex_off = d_texoff.as<long long>(); A.stg_off = d_stgoff.as<long long>();
  A.nlo = d_nlo.as<int32_t>(); A.nhalo = d_nhalo.as<int32_t>();
  const int halo_smem = 2 * gi::pow2_ceil(int(smax) * D) * 4;
  {
    auto fn = gi::k_halo<D, 1, false>;
    GALE_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit - 2048));  // the kernel has static shared memory too
    fn<<<nTiles, TB, halo_smem, st>>>(p.dT, p.d_tex.as<int32_t>(), A, kRefCap, nullptr, nullptr, d_flag.as<int>());
    GALE_CUDA(cudaGetLastError());
  }
  std::vector<int32_t> nlo, nhalo;
  if ((rc = download_vec(nlo, d_nlo.p, size_t(nTiles), st)) || (rc = download_vec(nhalo, d_nhalo.p, size_t(nTiles), st))) return rc;
  std::vector<long long> gid_off(nTiles);
  long long gido = 0, nlocm = 4;
  const int max_local = D == 4 ? gale::kMaxLocal4 : gale::kMaxLocal3;
  for (int i = 0; i < nTiles; ++i) {
    TileDesc& d = p.tiles[i];
    d.nlo = nlo[i];
    d.nloc = nhalo[i] + d.nrows;
    if (d.nloc > max_local) { fits = false; return GALE_OK; }
    d.gid_off = gid_off[i] = gido;
    gido += pad_to(d.nloc, 4);
    nlocm = std::max(nlocm, pad_to(d.nloc, 4));
  }
  // 8-bit local ids when every tile has at most 255 local vertices: half the staged bytes (HBM and shared
  // memory). 0xFF only pads the unused 4th entry of a triangle.
  p.cfg.lb = nlocm <= 255 ? 1 : 2;
  p.n_gid = size_t(gido) + 4;
  p.loc_bytes = size_t(stg) * 4 * p.cfg.lb + 64;
  if ((rc = p.d_gid.alloc(p.n_gid * 4)) || (rc = p.d_loc.alloc(p.loc_bytes)) || (rc = upload_vec(d_gidoff, gid_off, st))) return rc;
  A.gid_off = d_gidoff.as<long long>();
  {
    auto fn = p.cfg.lb == 1 ? gi::k_halo<D, 1, true> : gi::k_halo<D, 2, true>;
    GALE_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit - 2048));  // the kernel has static shared memory too
    fn<<<nTiles, TB, halo_smem, st>>>(p.dT, p.d_tex.as<int32_t>(), A, kRefCap, p.d_gid.as<int32_t>(), p.d_loc.p, d_flag.as<int>());
    GALE_CUDA(cudaGetLastError());
  }
  GALE_CUDA(cudaStreamSynchronize(st));
  p.cfg.smax = int(smax); p.cfg.sext = int(sextm); p.cfg.sint = int(sintm); p.cfg.nloc = int(nlocm);
  p.cfg.WT = int((smax + 31) / 32) | 1;
  p.cfg.WV = int((nlocm + 31) / 32) | 1;
  return GALE_OK;
}

// Sizing run (count mode of the dense kernel) over all tiles: exact VT / VV entry counts per tile.
// `fits` tells whether the count-mode shared memory fits at this tile size.
int run_sizing(Plan& p, cudaStream_t st, std::vector<long long>& stats, bool& fits) {
  const int D = p.dim + 1;
  fits = true;
  stats.assign(size_t(p.nTiles) * 4, 0);
  if (p.nTiles == 0) return GALE_OK;
  const SmemCfg c = cfg_for_mask(p.cfg, 3, true);
  const gale::SmemLayout lay = layout_for(D, c);
  if (lay.total > kSmemLimit) { fits = false; return GALE_OK; }
  DevMem b_tiles, b_stats, b_err;
  int rc;
  if ((rc = upload_vec(b_tiles, p.tiles, st)) || (rc = b_stats.alloc(stats.size() * 8)) || (rc = b_err.alloc(4))) return rc;
  GALE_CUDA(cudaMemsetAsync(b_err.p, 0, 4, st));
  DeviceMesh dm{};
  dm.T = p.dT;
  dm.first_tet = p.d_first_tet.as<int32_t>();
  dm.tiles = b_tiles.as<TileDesc>();
  dm.tex = p.d_tex.as<int32_t>();
  dm.gid = p.d_gid.as<int32_t>();
  dm.loc = p.d_loc.p;
  dm.err = b_err.as<int32_t>();
  KernelFn fn = kernel_for(D, p.NT, true, p.cfg.lb);
  GALE_CUDA(allow_max_smem(fn));
  gale::BatchParams P{};
  P.mask = 3u | gale::MODE_COUNT;
  gale::OutPtrs O{};
  O.stats = b_stats.as<long long>();
  fn<<<p.nTiles, p.NT, lay.total, st>>>(dm, P, c, lay, O);
  GALE_CUDA(cudaGetLastError());
  if ((rc = download_vec(stats, b_stats.p, stats.size(), st))) return rc;
  int err = 0;
  GALE_CUDA(cudaMemcpyAsync(&err, b_err.p, 4, cudaMemcpyDeviceToHost, st));
  GALE_CUDA(cudaStreamSynchronize(st));
  if (err) { g_last_error = "device guard fired during sizing: " + std::to_string(err); return GALE_ERR_WORKSPACE; }
  return GALE_OK;
}

// The initialization on the device: validation, I_T per vertex, the index of simplices
// by second vertex, tiles with their T_ex lists and local encodings, exact output sizes.
template <int D>
int analyse_device(Plan& p, const gale_mesh_desc_t& d, cudaStream_t st) {
  namespace gi = gale::init;
  const int TB = 256;
  int rc;
  DevMem d_flags;  // [0] not canonical, [1] gmax
  if ((rc = d_flags.alloc(8))) return rc;
  GALE_CUDA(cudaMemsetAsync(d_flags.p, 0, 8, st));
  if ((d.flags & (GALE_VALIDATE | GALE_VALIDATE_MANIFOLD)) && p.nT)
    gi::k_validate<D><<<blocks_for(p.nT, TB), TB, 0, st>>>(p.dT, p.nT, p.nV, d_flags.as<int>());
  {
    int bad = 0;
    GALE_CUDA(cudaMemcpyAsync(&bad, d_flags.p, 4, cudaMemcpyDeviceToHost, st));
    GALE_CUDA(cudaStreamSynchronize(st));
    if (bad) return GALE_ERR_NOT_CANONICAL;
  }
  if (d.flags & GALE_VALIDATE_MANIFOLD) {  // C4, optional: the facet sort runs on the host (slow path, opt-in)
    std::vector<int32_t> T;
    if ((rc = download_vec(T, p.dT, size_t(p.nT) * D, st))) return rc;
    if ((rc = validate_manifold<D>(p, T)) != GALE_OK) return rc;
  }
  // I_T per vertex; simplices grouped by second vertex
  DevMem d_scan, d_cursor;
  if ((rc = p.d_first_tet.alloc(size_t(p.nV + 2) * 4)) || (rc = p.d_opp_first.alloc(size_t(p.nV + 2) * 4)) ||
      (rc = p.d_opp_perm.alloc(size_t(std::max<long long>(p.nT, 1)) * 4)) ||
      (rc = d_scan.alloc((size_t(p.nV + 1) / gi::kScanChunk + 2) * 4)) || (rc = d_cursor.alloc(size_t(p.nV + 2) * 4)))
    return rc;
  gi::k_first_tet<D><<<blocks_for(p.nT + 1, TB), TB, 0, st>>>(p.dT, p.nT, p.nV, p.d_first_tet.as<int32_t>());
  GALE_CUDA(cudaMemsetAsync(p.d_opp_first.p, 0, size_t(p.nV + 2) * 4, st));
  if (p.nT) gi::k_second_count<D><<<blocks_for(p.nT, TB), TB, 0, st>>>(p.dT, p.nT, p.d_opp_first.as<int32_t>());
  GALE_CUDA(gi::exclusive_scan_i32(p.d_opp_first.as<int32_t>(), p.nV + 1, d_scan.as<int32_t>(), st));
  GALE_CUDA(cudaMemcpyAsync(d_cursor.p, p.d_opp_first.p, size_t(p.nV + 1) * 4, cudaMemcpyDeviceToDevice, st));
  if (p.nT) gi::k_second_fill<D><<<blocks_for(p.nT, TB), TB, 0, st>>>(p.dT, p.nT, d_cursor.as<int32_t>(), p.d_opp_perm.as<int32_t>());
  if (p.nV) gi::k_gmax<D><<<blocks_for(p.nV, TB), TB, 0, st>>>(p.d_first_tet.as<int32_t>(), p.d_opp_first.as<int32_t>(), p.nV, d_flags.as<int>() + 1);
  {  // I_T per cluster
    DevMem d_off, d_out;
    if ((rc = upload_vec(d_off, p.cl_off, st)) || (rc = d_out.alloc(size_t(p.nC + 1) * 4))) return rc;
    gi::k_gather<<<blocks_for(p.nC + 1, TB), TB, 0, st>>>(p.d_first_tet.as<int32_t>(), d_off.as<int32_t>(), p.nC + 1, d_out.as<int32_t>());
    if ((rc = download_vec(p.cl_t_lo, d_out.p, size_t(p.nC) + 1, st))) return rc;
    int g = 0;
    GALE_CUDA(cudaMemcpyAsync(&g, d_flags.as<int>() + 1, 4, cudaMemcpyDeviceToHost, st));
    GALE_CUDA(cudaStreamSynchronize(st));
    p.gmax = std::max(1, g);
  }
  d_cursor.release();

  int tv = d.tile_vertices > 0 ? std::min(d.tile_vertices, gale::kMaxTileVertices) : (d.dim == 3 ? 32 : 64);  // measured optima on configs 5 and 2
  std::vector<long long> stats;
  bool shrunk = false;
  for (;; tv = (tv + 1) / 2) {
    if (tv < 1) return GALE_ERR_UNSUPPORTED;
    const bool last = tv == 1;
    bool fits = true;
    if ((rc = build_tiles_device<D>(p, tv, st, fits)) != GALE_OK) return rc;
    if (fits && (rc = run_sizing(p, st, stats, fits)) != GALE_OK) return rc;
    if (fits) {
      long long vt_max = 1, vv_max = 1, tbl_max = 4;
      for (int i = 0; i < p.nTiles; ++i) {
        vt_max = std::max(vt_max, stats[i * 4 + 0]);
        vv_max = std::max(vv_max, stats[i * 4 + 1]);
        tbl_max = std::max(tbl_max, stats[i * 4 + 0] + (long long)(D - 2) * p.tiles[i].s_int);
      }
      p.cfg.vt_max = int(pad_to(vt_max, 8));
      p.cfg.vv_max = int(pad_to(vv_max, 8));
      p.cfg.tbl = int(pad_to(tbl_max, 4));
      p.smem_bytes = layout_for(D, p.cfg).total;
      fits = vt_max <= gale::kMaxNnz16 && vv_max <= gale::kMaxNnz16 && p.smem_bytes <= kSmemLimit;
    }
    // automatic tile size: tiles whose vertices are scattered in the mesh (graded or irregular meshes) need
    // large per-block capacities and leave few resident blocks; 24-vertex tiles measured +10 % on config 4
    // (8.1 -> 8.9 G tets/s) against 32
    if (fits && d.tile_vertices == 0 && !shrunk && tv == 32 && D == 4 && p.smem_bytes > 28 * 1024) {
      shrunk = true;
      tv = 47;  // the loop step turns it into 24
      continue;
    }
    if (fits) break;
    if (last) { g_last_error = "a single vertex star exceeds the kernels' shared-memory limits"; return GALE_ERR_UNSUPPORTED; }
  }
  {  // can the walk kernel run these tiles?
    // as many slots as the largest group has records: when a record is placed at most gmax - 1 slots are
    // taken, so the probe always meets an empty slot or its key; every interior facet is recorded twice, so
    // the usual load is about 0.5 (the tables are bank-conflict free, re-probes are cheap; the 1 KB saved
    // per block buys two more resident blocks)
    p.cfg.hs = std::max(8, p.gmax);
    p.w_NT = walk_threads_for_tile(p.tv);
    p.w_smem = walk_layout_for(D, walk_cfg_for_mask(p.cfg, 7)).total;
    p.walk_ok = p.tv <= 256 && p.w_smem <= kSmemLimit && p.cfg.smax < 32768 && p.cfg.vt_max < 65536;
  }
  // per-tile output placement inside its cluster, per-cluster sizes
  p.cl_vt.assign(p.nC, 0);
  p.cl_vv.assign(p.nC, 0);
  for (int c = 0; c < p.nC; ++c) {
    long long vt = 0, vv = 0;
    for (int i = p.cl_tile_begin[c]; i < p.cl_tile_begin[c + 1]; ++i) {
      TileDesc& t = p.tiles[i];
      if (vt > INT32_MAX || vv > INT32_MAX) return GALE_ERR_UNSUPPORTED;
      t.vt_rel = int32_t(vt); t.vv_rel = int32_t(vv);
      t.vt_nnz = int32_t(stats[i * 4 + 0]); t.vv_nnz = int32_t(stats[i * 4 + 1]);
      vt += t.vt_nnz; vv += t.vv_nnz;
    }
    p.cl_vt[c] = vt; p.cl_vv[c] = vv;
    p.vt_total += vt; p.vv_total += vv;
    p.max_rows = std::max<long long>(p.max_rows, p.cl_off[c + 1] - p.cl_off[c]);
    p.max_vt = std::max(p.max_vt, vt);
    p.max_vv = std::max(p.max_vv, vv);
    p.max_tt = std::max<long long>(p.max_tt, p.cl_t_lo[c + 1] - p.cl_t_lo[c]);
  }
  return GALE_OK;
}

int analyse(const gale_mesh_desc_t& d, cudaStream_t st, std::unique_ptr<Plan>& out) {
  const auto t0 = std::chrono::steady_clock::now();
  auto p = std::make_unique<Plan>();
  p->dT = d.d_simplices; p->dim = d.dim; p->nV = d.num_vertices; p->nC = d.num_clusters; p->nT = d.num_simplices;
  p->tv_req = d.tile_vertices; p->flags = d.flags;
  p->maxB = d.max_batch_clusters; p->queue_depth = d.queue_depth; p->device_ring = d.device_ring;
  p->cl_off.assign(d.h_cluster_offsets, d.h_cluster_offsets + d.num_clusters + 1);
  if (p->cl_off.front() != 0 || p->cl_off.back() != p->nV) return GALE_ERR_INVALID_ARG;
  for (int c = 0; c < p->nC; ++c)
    if (p->cl_off[c] > p->cl_off[c + 1]) return GALE_ERR_INVALID_ARG;
  const int rc = d.dim == 3 ? analyse_device<4>(*p, d, st) : analyse_device<3>(*p, d, st);
  if (rc != GALE_OK) return rc;
  p->analyse_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  out = std::move(p);
  return GALE_OK;
}

int check_desc(const gale_mesh_desc_t* d) {
  if (!d || (d->dim != 2 && d->dim != 3) || d->num_vertices < 0 || d->num_simplices < 0 || d->num_clusters < 0 ||
      !d->h_cluster_offsets || (d->num_simplices > 0 && !d->d_simplices) || d->max_batch_clusters < 1 ||
      d->queue_depth < 0 || d->device_ring < 0 || d->tile_vertices < 0 || d->num_simplices >= (1LL << 31) - 1 ||
      (d->flags & ~uint32_t(GALE_VALIDATE | GALE_VALIDATE_MANIFOLD | GALE_STREAM_ORDERED | GALE_KERNEL_DENSE | GALE_KERNEL_WALK | GALE_STAGE_FROM_T | GALE_WITH_EDGES | GALE_WITH_FACETS | GALE_WITH_COBOUNDARY)) ||
      ((d->flags & GALE_WITH_FACETS) && d->dim != 3) ||
      ((d->flags & GALE_WITH_COBOUNDARY) && (d->flags & (GALE_WITH_EDGES | GALE_WITH_FACETS)) != (GALE_WITH_EDGES | GALE_WITH_FACETS)) ||
      (d->flags & (GALE_KERNEL_DENSE | GALE_KERNEL_WALK)) == (GALE_KERNEL_DENSE | GALE_KERNEL_WALK) ||
      (d->flags & (GALE_STAGE_FROM_T | GALE_KERNEL_WALK)) == (GALE_STAGE_FROM_T | GALE_KERNEL_WALK))  // the walk kernel cannot stage from T
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
  L.first_tet = take(size_t(p.nV + 1) * 4);
  L.opp_first = take(size_t(p.nV + 1) * 4);
  L.opp_perm = take(size_t(p.nT) * 4);
  L.cl_tile_begin = take(p.cl_tile_begin.size() * 4);
  L.tiles = take(p.tiles.size() * sizeof(TileDesc));
  L.tex = take(p.n_tex * 4);
  L.gid = take(p.n_gid * 4);
  L.loc = take(p.loc_bytes);
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
  long long rows = 0, vt_nnz = 0, vv_nnz = 0, tt_rows = 0, vf_nnz = 0;
  std::vector<int32_t> e_row_begin, f_row_begin;
  long long cob_nnz[3] = {0, 0, 0};
  uint32_t eff_mask = 0;  // what the batch kernel computed (VE implies VV, VF implies VT)
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
  static constexpr int kMaxLaunchStreams = 2;
  int n_launch = 2;  // streams in use (3, 4 and 8 measured flat on configs 4 and 5)
  cudaStream_t launch[kMaxLaunchStreams] = {};
  int32_t* h_err = nullptr;  // mapped pinned; the kernels write guard codes here
  std::atomic<long long> submitted{0}, popped{0};
  size_t workspace_used = 0, index_bytes = 0;
  double create_ms = 0;
  float tune_ms[2] = {0.f, 0.f};
  // edges / triangles (GALE_WITH_EDGES / GALE_WITH_FACETS): library-owned device memory
  DevMem d_cl_off, d_e_first, d_e_hi, d_f_first, d_f_bc;
  long long nE = 0, nF = 0;
  // VF (GALE_WITH_FACETS) and EF / ET / FT (GALE_WITH_COBOUNDARY), indexed by gale::sub::COB_* (VF = 3)
  DevMem d_tile_cob_rel[4];             // first entry of a tile inside its cluster
  std::vector<long long> cl_cob[4];     // entries per cluster
  std::vector<int32_t> cl_e0, cl_f0;    // [nC+1] I_E / I_F at the cluster boundaries
  int rows_cap_e = 0, rows_cap_f = 0;   // most edges / triangles of a tile
  int star_t = 1, star_f = 1;           // largest stars of k_star: |VT(v)|; triangles at a vertex
  int fblock_max = 1, fstar_tile = 4;   // longest block of F; most triangles at the vertices of a tile
  bool cob_ready = false;
  gale::sub::SubIndex sub{};  // sample-batch time of the dense / walk kernel at create (0 = not timed)
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

// Edges / triangles (E, I_E, F, I_F "generated only when the edge or
// triangle information is explicitly needed"). Built with the handle's own hot path: E from the upper part
// of the VV rows of every cluster, F from the facet groups of the vertices; the exact VF sizes per tile come
// from a counting sweep over the VT rows.
template <class Fn>
int sweep_batches(gale_mesh* m, uint32_t mask, cudaStream_t st, Fn&& per_batch) {
  const Plan& p = *m->plan;
  std::vector<int32_t> ids;
  for (int c0 = 0; c0 < p.nC; c0 += m->maxB) {
    const int n = std::min(m->maxB, p.nC - c0);
    ids.resize(size_t(n));
    for (int i = 0; i < n; ++i) ids[size_t(i)] = c0 + i;
    int rc = gale_cluster_batch_compute(m, mask, ids.data(), n, st);
    gale_batch_view_t v;
    if (rc == GALE_OK) rc = gale_queue_pop(m, &v, -1);
    if (rc != GALE_OK) return rc;
    rc = per_batch(*m->slots[size_t(v.slot)], c0, n);  // the slot's DEVICE copy is complete (pop waited for it)
    GALE_CUDA(cudaStreamSynchronize(st));
    const int rc2 = gale_queue_release(m, &v);
    if (rc != GALE_OK) return rc;
    if (rc2 != GALE_OK) return rc2;
  }
  m->submitted.store(0); m->popped.store(0);  // these batches were the library's own
  return GALE_OK;
}

// ---- VF / EF / ET / FT launches (gale_sub.cuh: k_star) ---------------------------------------------------------
constexpr int kStarWarps = 8;
struct StarCfg { gale::sub::StarDims d; gale::sub::StarLayout lay; int smem; };
StarCfg star_cfg(const gale_mesh* m, int kind) {
  namespace gs = gale::sub;
  const Plan& p = *m->plan;
  const bool from_vt = kind == gs::COB_ET || kind == gs::COB_FT;
  StarCfg c;
  c.d.tv = p.tv;
  c.d.rows_cap = kind == gs::COB_VF ? 0 : (kind == gs::COB_FT ? m->rows_cap_f : m->rows_cap_e);
  c.d.src_cap = std::max(4, from_vt ? p.cfg.vt_max : p.cfg.vv_max);  // the tile capacities of the batch kernel
  c.d.W = kind == gs::COB_VF ? 0 : ((from_vt ? m->star_t : m->star_f) + 31) / 32;
  c.d.Wf = from_vt ? 0 : (m->fblock_max + 31) / 32;
  c.d.fstar_cap = kind == gs::COB_EF ? m->fstar_tile : 0;
  c.lay = gs::make_star_layout(kind, c.d);
  c.smem = c.lay.total * 4;
  return c;
}
// src = the batch's VT rows (ET, FT) or VV rows (EF, VF)
template <bool COUNT>
void launch_star(const gale_mesh* m, int kind, int grid, const gale::sub::CobParams& V, const int32_t* src_off,
                 const int32_t* src_idx, int32_t* out_off, int32_t* out_idx, int32_t* stats, int32_t* stats_max, cudaStream_t st) {
  namespace gs = gale::sub;
  const StarCfg c = star_cfg(m, kind);
  const int32_t* rel = COUNT ? nullptr : m->d_tile_cob_rel[kind].as<int32_t>();
#define GALE_STAR(K) gs::k_star<K, COUNT><<<grid, kStarWarps * 32, c.smem, st>>>(m->dm, m->sub, V, c.d, c.lay, rel, src_off, src_idx, out_off, out_idx, stats, stats_max)
  switch (kind) {
    case gs::COB_ET: GALE_STAR(gs::COB_ET); break;
    case gs::COB_FT: GALE_STAR(gs::COB_FT); break;
    case gs::COB_EF: GALE_STAR(gs::COB_EF); break;
    default: GALE_STAR(gs::COB_VF); break;
  }
#undef GALE_STAR
}
int star_allow_smem() {
  // set on every create, for the device that is current: a cached "done" would leave a second device (or a new
  // context) without the attribute, and k_star launches with more than 48 KB would fail there
  namespace gs = gale::sub;
#define GALE_ATTR(K) GALE_CUDA(cudaFuncSetAttribute(gs::k_star<K, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit - 2048)); \
                     GALE_CUDA(cudaFuncSetAttribute(gs::k_star<K, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit - 2048))
  GALE_ATTR(gs::COB_ET); GALE_ATTR(gs::COB_FT); GALE_ATTR(gs::COB_EF); GALE_ATTR(gs::COB_VF);
#undef GALE_ATTR
  return GALE_OK;
}

// Exact sizes of the relations in `kinds` (bits 1 << COB_*): one counting sweep over the batches with the source
// relations `src_mask`; fills cl_cob, d_tile_cob_rel and (VF) the star sizes of EF.
int size_star_relations(gale_mesh* m, cudaStream_t st, uint32_t kinds, uint32_t src_mask) {
  namespace gs = gale::sub;
  const Plan& p = *m->plan;
  int rc;
  if ((rc = star_allow_smem())) return rc;
  DevMem d_stats[4], d_max;
  if ((rc = d_max.alloc(16))) return rc;
  GALE_CUDA(cudaMemsetAsync(d_max.p, 0, 16, st));
  for (int k = 0; k < 4; ++k) {
    if (!(kinds >> k & 1u)) continue;
    if ((rc = d_stats[k].alloc(size_t(std::max(p.nTiles, 1)) * 4))) return rc;
    if (star_cfg(m, k).smem > kSmemLimit - 2048) { g_last_error = "a vertex star or a tile is too large for the VF / EF / ET / FT kernels"; return GALE_ERR_UNSUPPORTED; }
  }
  rc = sweep_batches(m, src_mask, st, [&](const Slot& s, int, int n) -> int {
    const int32_t* vt_off = reinterpret_cast<const int32_t*>(s.dev + s.used.vt_off);
    const int32_t* vt_idx = reinterpret_cast<const int32_t*>(s.dev + s.used.vt_idx);
    const int32_t* vv_off = reinterpret_cast<const int32_t*>(s.dev + s.used.vv_off);
    const int32_t* vv_idx = reinterpret_cast<const int32_t*>(s.dev + s.used.vv_idx);
    for (int b = 0; b < n; b += gale::kMaxBatch) {
      const int nb = std::min(gale::kMaxBatch, n - b);
      gs::CobParams V{};
      V.n_clusters = nb;
      for (int i = 0; i < nb; ++i) {
        const int c = s.ids[size_t(b + i)];
        V.tile_prefix[i + 1] = V.tile_prefix[i] + (p.cl_tile_begin[c + 1] - p.cl_tile_begin[c]);
        V.cluster[i] = c;
        V.src_row_base[i] = s.row_begin[size_t(b + i)];
      }
      const int grid = V.tile_prefix[nb];
      if (grid <= 0) continue;
      {
        const int per = V.tile_prefix[1];
        bool uniform = per > 0;
        for (int i = 0; i < nb && uniform; ++i) uniform = V.tile_prefix[i + 1] - V.tile_prefix[i] == per;
        V.uniform_tiles = uniform ? per : 0;
      }
      for (int k = 0; k < 4; ++k) {
        if (!(kinds >> k & 1u)) continue;
        const bool from_vt = k == gs::COB_ET || k == gs::COB_FT;
        launch_star<true>(m, k, grid, V, from_vt ? vt_off : vv_off, from_vt ? vt_idx : vv_idx, nullptr, nullptr,
                          d_stats[k].as<int32_t>(), d_max.as<int32_t>() + k, st);
      }
    }
    GALE_CUDA(cudaGetLastError());
    return int(GALE_OK);
  });
  if (rc != GALE_OK) return rc;
  int32_t vmax[4] = {0, 0, 0, 0};
  GALE_CUDA(cudaMemcpyAsync(vmax, d_max.p, 16, cudaMemcpyDeviceToHost, st));
  GALE_CUDA(cudaStreamSynchronize(st));
  for (int k = 0; k < 4; ++k) {
    if (!(kinds >> k & 1u)) continue;
    std::vector<int32_t> stats, rel(size_t(std::max(p.nTiles, 1)), 0);
    if ((rc = download_vec(stats, d_stats[k].p, size_t(p.nTiles), st))) return rc;
    m->cl_cob[k].assign(size_t(p.nC), 0);
    const long long per_vt = k == gs::COB_EF ? 6LL : 3LL;  // the per-cluster bounds of slot_capacity_layout
    for (int c = 0; c < p.nC; ++c) {
      long long acc = 0;
      for (int i = p.cl_tile_begin[c]; i < p.cl_tile_begin[c + 1]; ++i) { rel[size_t(i)] = int32_t(acc); acc += stats[size_t(i)]; }
      if (acc > per_vt * (k == gs::COB_VF ? p.cl_vt[size_t(c)] : p.max_vt) || acc >= (1LL << 31) - 1) { g_last_error = "a relation exceeds its slot bound"; return GALE_ERR_UNSUPPORTED; }
      m->cl_cob[k][size_t(c)] = acc;
    }
    if (k == gs::COB_VF) {  // the star of EF: the triangles at a vertex / at the vertices of a tile
      m->star_f = std::max(1, int(vmax[k]));
      m->fstar_tile = 4;
      for (int i = 0; i < p.nTiles; ++i) m->fstar_tile = std::max(m->fstar_tile, int(stats[size_t(i)]));
    }
    if ((rc = upload_vec(m->d_tile_cob_rel[k], rel, st))) return rc;
  }
  GALE_CUDA(cudaStreamSynchronize(st));
  return GALE_OK;
}

int build_sub_index(gale_mesh* m, cudaStream_t st) {
  namespace gs = gale::sub;
  namespace gi = gale::init;
  const Plan& p = *m->plan;
  const int TB = 256;
  int rc;
  if ((rc = upload_vec(m->d_cl_off, p.cl_off, st))) return rc;
  m->sub.cl_off = m->d_cl_off.as<int32_t>();
  DevMem d_scan;
  if ((rc = d_scan.alloc((size_t(p.nV + 1) / gi::kScanChunk + 2) * 4))) return rc;
  auto for_chunks = [&](const Slot& s, int n, auto&& fn) {  // <= kMaxBatch clusters per descriptor
    for (int b = 0; b < n; b += gale::kMaxBatch) {
      const int nb = std::min(gale::kMaxBatch, n - b);
      gs::BatchRows B{};
      B.n_clusters = nb;
      for (int i = 0; i <= nb; ++i) B.row_base[i] = s.row_begin[size_t(b + i)];
      for (int i = 0; i < nb; ++i) B.cluster[i] = s.ids[size_t(b + i)];
      const int rows = B.row_base[nb] - B.row_base[0];
      if (rows > 0) fn(B, rows);
    }
  };
  if (p.flags & GALE_WITH_EDGES) {
    if ((rc = m->d_e_first.alloc(size_t(p.nV + 2) * 4))) return rc;
    GALE_CUDA(cudaMemsetAsync(m->d_e_first.p, 0, size_t(p.nV + 2) * 4, st));
    int32_t* first = m->d_e_first.as<int32_t>();
    rc = sweep_batches(m, GALE_REL_VV, st, [&](const Slot& s, int, int n) -> int {
      const int32_t* off = reinterpret_cast<const int32_t*>(s.dev + s.used.vv_off);
      const int32_t* idx = reinterpret_cast<const int32_t*>(s.dev + s.used.vv_idx);
      for_chunks(s, n, [&](const gs::BatchRows& B, int rows) {
        gs::k_upper_edges<true><<<blocks_for(rows, TB), TB, 0, st>>>(B, m->sub.cl_off, off, idx, first, nullptr);
      });
      GALE_CUDA(cudaGetLastError());
      return int(GALE_OK);
    });
    if (rc != GALE_OK) return rc;
    GALE_CUDA(gi::exclusive_scan_i32(first, p.nV + 1, d_scan.as<int32_t>(), st));
    int nE = 0;
    GALE_CUDA(cudaMemcpyAsync(&nE, first + p.nV, 4, cudaMemcpyDeviceToHost, st));
    GALE_CUDA(cudaStreamSynchronize(st));
    m->nE = nE;
    if ((rc = m->d_e_hi.alloc(size_t(std::max(nE, 1)) * 4 + 64))) return rc;
    int32_t* hi = m->d_e_hi.as<int32_t>();
    rc = sweep_batches(m, GALE_REL_VV, st, [&](const Slot& s, int, int n) -> int {
      const int32_t* off = reinterpret_cast<const int32_t*>(s.dev + s.used.vv_off);
      const int32_t* idx = reinterpret_cast<const int32_t*>(s.dev + s.used.vv_idx);
      for_chunks(s, n, [&](const gs::BatchRows& B, int rows) {
        gs::k_upper_edges<false><<<blocks_for(rows, TB), TB, 0, st>>>(B, m->sub.cl_off, off, idx, first, hi);
      });
      GALE_CUDA(cudaGetLastError());
      return int(GALE_OK);
    });
    if (rc != GALE_OK) return rc;
    m->sub.e_first = first;
    m->sub.e_hi = hi;
  }
  if (p.flags & GALE_WITH_FACETS) {
    const int warps = 4, cap = gi::pow2_ceil(std::max(p.gmax, 1));
    const int smem = warps * cap * 8;
    if (smem > kSmemLimit - 2048) { g_last_error = "a vertex has too many facets for the triangle enumeration"; return GALE_ERR_UNSUPPORTED; }
    if ((rc = m->d_f_first.alloc(size_t(p.nV + 2) * 4))) return rc;
    GALE_CUDA(cudaMemsetAsync(m->d_f_first.p, 0, size_t(p.nV + 2) * 4, st));
    int32_t* first = m->d_f_first.as<int32_t>();
    GALE_CUDA(cudaFuncSetAttribute(gs::k_triangles<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit - 2048));
    GALE_CUDA(cudaFuncSetAttribute(gs::k_triangles<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit - 2048));
    const int grid = blocks_for(p.nV, warps);
    if (p.nV) gs::k_triangles<true><<<grid, warps * 32, smem, st>>>(m->dm.T, m->dm.first_tet, m->dm.opp_first, m->dm.opp_perm, p.nV, cap, first, nullptr);
    GALE_CUDA(cudaGetLastError());
    GALE_CUDA(gi::exclusive_scan_i32(first, p.nV + 1, d_scan.as<int32_t>(), st));
    int nF = 0;
    GALE_CUDA(cudaMemcpyAsync(&nF, first + p.nV, 4, cudaMemcpyDeviceToHost, st));
    GALE_CUDA(cudaStreamSynchronize(st));
    m->nF = nF;
    if ((rc = m->d_f_bc.alloc(size_t(std::max(nF, 1)) * 8 + 64))) return rc;
    if (p.nV) gs::k_triangles<false><<<grid, warps * 32, smem, st>>>(m->dm.T, m->dm.first_tet, m->dm.opp_first, m->dm.opp_perm, p.nV, cap, first, m->d_f_bc.as<int2>());
    GALE_CUDA(cudaGetLastError());
    m->sub.f_first = first;
    m->sub.f_bc = m->d_f_bc.as<int2>();
    // sizing of VF: the largest |VT(v)| (star capacities), then the exact entries per tile
    DevMem d_max;
    if ((rc = d_max.alloc(4))) return rc;
    GALE_CUDA(cudaMemsetAsync(d_max.p, 0, 4, st));
    rc = sweep_batches(m, GALE_REL_VT, st, [&](const Slot& s, int, int) -> int {
      const int32_t* off = reinterpret_cast<const int32_t*>(s.dev + s.used.vt_off);
      if (s.rows > 0) gs::k_max_row<<<blocks_for(s.rows, TB), TB, 0, st>>>(off, int(s.rows), d_max.as<int>());
      GALE_CUDA(cudaGetLastError());
      return int(GALE_OK);
    });
    if (rc != GALE_OK) return rc;
    int maxdeg = 0;
    GALE_CUDA(cudaMemcpyAsync(&maxdeg, d_max.p, 4, cudaMemcpyDeviceToHost, st));
    GALE_CUDA(cudaStreamSynchronize(st));
    m->star_t = std::max(maxdeg, 1);
    {  // longest block of F
      GALE_CUDA(cudaMemsetAsync(d_max.p, 0, 4, st));
      if (p.nV) gs::k_max_row<<<blocks_for(p.nV, TB), TB, 0, st>>>(first, p.nV, d_max.as<int>());
      int mx = 0;
      GALE_CUDA(cudaMemcpyAsync(&mx, d_max.p, 4, cudaMemcpyDeviceToHost, st));
      GALE_CUDA(cudaStreamSynchronize(st));
      m->fblock_max = std::max(mx, 1);
    }
    if ((rc = size_star_relations(m, st, 1u << gs::COB_VF, GALE_REL_VV))) return rc;
  }
  if (p.flags & GALE_WITH_COBOUNDARY) {
    // EF / ET / FT: rows per cluster and per tile from I_E / I_F at their boundaries, then exact entries per
    // tile from a counting sweep over the VT / VV rows
    std::vector<int32_t> tile_v(size_t(p.nTiles) + 1, p.nV), tile_e, tile_f;
    for (int i = 0; i < p.nTiles; ++i) tile_v[size_t(i)] = p.tiles[size_t(i)].v_lo;
    {
      DevMem d_idx, d_out;
      auto gather = [&](const std::vector<int32_t>& idx, const int32_t* src, std::vector<int32_t>& out) -> int {
        int r2;
        if ((r2 = upload_vec(d_idx, idx, st)) || (r2 = d_out.alloc(idx.size() * 4))) return r2;
        gi::k_gather<<<blocks_for((long long)idx.size(), TB), TB, 0, st>>>(src, d_idx.as<int32_t>(), int(idx.size()), d_out.as<int32_t>());
        return download_vec(out, d_out.p, idx.size(), st);
      };
      if ((rc = gather(p.cl_off, m->sub.e_first, m->cl_e0)) || (rc = gather(p.cl_off, m->sub.f_first, m->cl_f0)) ||
          (rc = gather(tile_v, m->sub.e_first, tile_e)) || (rc = gather(tile_v, m->sub.f_first, tile_f)))
        return rc;
    }
    // tiles are numbered cluster by cluster with ascending v_lo, but empty clusters own no tile: rows of tile i end
    // where its vertices end
    m->rows_cap_e = m->rows_cap_f = 4;
    {
      std::vector<int32_t> vend(size_t(p.nTiles));
      for (int i = 0; i < p.nTiles; ++i) vend[size_t(i)] = p.tiles[size_t(i)].v_lo + p.tiles[size_t(i)].nrows;
      std::vector<int32_t> e_end, f_end;
      DevMem d_idx, d_out;
      auto gather2 = [&](const int32_t* src, std::vector<int32_t>& out) -> int {
        int r2;
        if ((r2 = upload_vec(d_idx, vend, st)) || (r2 = d_out.alloc(std::max<size_t>(vend.size(), 1) * 4))) return r2;
        if (!vend.empty()) gi::k_gather<<<blocks_for((long long)vend.size(), TB), TB, 0, st>>>(src, d_idx.as<int32_t>(), int(vend.size()), d_out.as<int32_t>());
        return download_vec(out, d_out.p, vend.size(), st);
      };
      if ((rc = gather2(m->sub.e_first, e_end)) || (rc = gather2(m->sub.f_first, f_end))) return rc;
      for (int i = 0; i < p.nTiles; ++i) {
        m->rows_cap_e = std::max(m->rows_cap_e, e_end[size_t(i)] - tile_e[size_t(i)]);
        m->rows_cap_f = std::max(m->rows_cap_f, f_end[size_t(i)] - tile_f[size_t(i)]);
      }
    }
    if ((rc = size_star_relations(m, st, (1u << gs::COB_ET) | (1u << gs::COB_FT) | (1u << gs::COB_EF), GALE_REL_VT | GALE_REL_VV))) return rc;
    m->cob_ready = true;
  }
  return GALE_OK;
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
  auto put = [&](size_t at, const void* src, size_t bytes, cudaMemcpyKind kind) -> int {
    if (bytes) GALE_CUDA(cudaMemcpyAsync(base + at, src, bytes, kind, st));
    return GALE_OK;
  };
  const cudaMemcpyKind D2D = cudaMemcpyDeviceToDevice, H2D = cudaMemcpyHostToDevice;
  int rc;
  if ((rc = put(IL.first_tet, p->d_first_tet.p, size_t(p->nV + 1) * 4, D2D)) ||
      (rc = put(IL.opp_first, p->d_opp_first.p, size_t(p->nV + 1) * 4, D2D)) ||
      (rc = put(IL.opp_perm, p->d_opp_perm.p, size_t(p->nT) * 4, D2D)) ||
      (rc = put(IL.cl_tile_begin, p->cl_tile_begin.data(), p->cl_tile_begin.size() * 4, H2D)) ||
      (rc = put(IL.tiles, p->tiles.data(), p->tiles.size() * sizeof(TileDesc), H2D)) ||
      (rc = put(IL.tex, p->d_tex.p, p->n_tex * 4, D2D)) || (rc = put(IL.gid, p->d_gid.p, p->n_gid * 4, D2D)) ||
      (rc = put(IL.loc, p->d_loc.p, p->loc_bytes, D2D)))
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
  // the library's own copy of the index is dropped once it sits in the workspace
  GALE_CUDA(cudaStreamSynchronize(st));
  p->d_first_tet.release(); p->d_opp_first.release(); p->d_opp_perm.release();
  p->d_tex.release(); p->d_gid.release(); p->d_loc.release();

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
    for (int i = 0; i < m->n_launch; ++i) GALE_CUDA(cudaStreamCreateWithFlags(&m->launch[i], cudaStreamNonBlocking));
  GALE_CUDA(allow_max_smem(kernel_for(m->D, p->NT, false, p->cfg.lb)));
  if (p->walk_ok) {
    GALE_CUDA(cudaFuncSetAttribute(walk_kernel_for(m->D, p->w_NT, p->cfg.lb, false), cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit));
    GALE_CUDA(cudaFuncSetAttribute(walk_kernel_for(m->D, p->w_NT, p->cfg.lb, true), cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit));
  }
  uint32_t force = p->flags & (GALE_KERNEL_DENSE | GALE_KERNEL_WALK);
  if (p->flags & GALE_STAGE_FROM_T) force = GALE_KERNEL_DENSE;  // only the dense kernel can stage from T: the flag selects it
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
  if (m->plan->flags & (GALE_WITH_EDGES | GALE_WITH_FACETS)) {
    const int rc3 = build_sub_index(m, st);
    if (rc3 != GALE_OK) return rc3;
  }
  m->create_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count() + m->plan->analyse_ms;
  guard.m = nullptr;
  *out = m;
  return GALE_OK;
}
}  // namespace

// ---- scratch of gale_canonicalize_static (include/gale.h) ----------------------------------------------------
// Everything the radix sort of gale_canon.cuh needs besides the caller's input and output, for callers that
// cannot allocate device memory (an in-situ analysis inside a host application whose pool owns the whole GPU,
// a loop that cannot take cudaMalloc's device-wide synchronisation). The array is part of the library image:
// every GPU that loads this library's code holds these ~25 MiB until the process exits. It is never
// initialised by the library beyond what a call writes, and it keeps the previous call's contents.
// NOTE for host code in this file: `g_canon_static_scratch` names a host-side stand-in of the symbol, not device
// memory — kernels must be given the address canon_static_base() obtains with cudaGetSymbolAddress.
namespace {
constexpr long long kCanonStaticMaxN = GALE_CANON_STATIC_MAX_SIMPLICES;
constexpr int kCanonStaticMaxSeg = (int)(kCanonStaticMaxN / gale::canon::kSeg);
constexpr size_t kCsT1 = 0;                                                   // int32[maxN * 4]  second row buffer
constexpr size_t kCsP0 = kCsT1 + size_t(kCanonStaticMaxN) * 16;               // int32[maxN]      permutation (no d_perm_out)
constexpr size_t kCsP1 = kCsP0 + size_t(kCanonStaticMaxN) * 4;                // int32[maxN]      permutation, other side
constexpr size_t kCsCounts = kCsP1 + size_t(kCanonStaticMaxN) * 4;            // int32[256 * maxSeg]
constexpr size_t kCsScan = kCsCounts + size_t(gale::canon::kDigits) * kCanonStaticMaxSeg * 4;   // chunk sums of the scan
constexpr size_t kCsBad = kCsScan + 256;                                      // int: the error flag, cleared per call
constexpr size_t kCsTotal = kCsBad + 256;
static_assert(kCanonStaticMaxN % gale::canon::kSeg == 0, "whole segments");
static_assert((size_t(gale::canon::kDigits) * kCanonStaticMaxSeg / gale::init::kScanChunk + 2) * 4 <= 256, "scan sums fit their slot");
static_assert(kCsTotal == GALE_CANON_STATIC_SCRATCH_BYTES, "gale.h states the size of the static scratch");
static_assert(kCsP0 % 256 == 0 && kCsP1 % 256 == 0 && kCsCounts % 256 == 0 && kCsScan % 256 == 0, "256-byte aligned parts");
}  // namespace

static __device__ __align__(256) unsigned char g_canon_static_scratch[kCsTotal];

namespace {
constexpr int kCanonStaticMaxDevices = 64;
std::mutex g_canon_static_mutex;                                  // set-up table AND the calls themselves (one array per device)
unsigned char* g_canon_static_ptr[kCanonStaticMaxDevices] = {};   // device address of the array, per device ordinal

// Device address of the scratch array on the CURRENT device; resolved once per device (the caller holds the
// mutex). No allocation: cudaGetSymbolAddress only reports where the module's global lives.
int canon_static_base(unsigned char** out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    g_last_error = "no CUDA device";
    return GALE_ERR_UNSUPPORTED;
  }
  if (dev < 0 || dev >= kCanonStaticMaxDevices) {
    g_last_error = "gale_canonicalize_static: device ordinal " + std::to_string(dev) + " beyond the " +
                   std::to_string(kCanonStaticMaxDevices) + " this entry keeps addresses for";
    return GALE_ERR_UNSUPPORTED;
  }
  if (!g_canon_static_ptr[dev]) {
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10) {
      cudaGetLastError();
      g_last_error = "device is not sm_100";
      return GALE_ERR_UNSUPPORTED;
    }
    unsigned char* p = nullptr;
    GALE_CUDA(cudaGetSymbolAddress((void**)&p, g_canon_static_scratch));
    if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) {
      g_last_error = "gale_canonicalize_static: the scratch array has no usable device address";
      return GALE_ERR_CUDA;
    }
    g_canon_static_ptr[dev] = p;
  }
  *out = g_canon_static_ptr[dev];
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

int32_t gale_canonicalize(int32_t dim, int64_t num_simplices, int32_t num_vertices, const int32_t* d_simplices_in,
                          int32_t* d_simplices_out, int32_t* d_perm_out, void* cuda_stream) {
  namespace gc = gale::canon;
  if ((dim != 2 && dim != 3) || num_simplices < 0 || num_simplices > 0x7FFFFFFFll || num_vertices <= 0) return GALE_ERR_INVALID_ARG;
  if (num_simplices > 0 && (!d_simplices_in || !d_simplices_out || d_simplices_in == d_simplices_out)) return GALE_ERR_INVALID_ARG;
  int rc = check_device();
  if (rc != GALE_OK) return rc;
  if (num_simplices == 0) return GALE_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int D = dim + 1;
  const long long n = num_simplices;
  const int nseg = (int)((n + gc::kSeg - 1) / gc::kSeg);
  const size_t n_counts = size_t(gc::kDigits) * nseg;
  DevMem d_T1, d_p0, d_p1, d_counts, d_scratch, d_bad;
  if ((rc = d_T1.alloc(size_t(n) * D * 4)) || (rc = d_p1.alloc(size_t(n) * 4)) || (rc = d_counts.alloc(n_counts * 4)) ||
      (rc = d_scratch.alloc((n_counts / gale::init::kScanChunk + 2) * 4)) || (rc = d_bad.alloc(4)))
    return rc;
  if (!d_perm_out && (rc = d_p0.alloc(size_t(n) * 4))) return rc;
  gc::Buffers B;
  B.T[0] = d_simplices_out; B.T[1] = d_T1.as<int32_t>();
  B.perm[0] = d_perm_out ? d_perm_out : d_p0.as<int32_t>(); B.perm[1] = d_p1.as<int32_t>();
  B.counts = d_counts.as<int32_t>(); B.scratch = d_scratch.as<int32_t>(); B.bad = d_bad.as<int>();
  GALE_CUDA(cudaMemsetAsync(B.bad, 0, 4, st));
  GALE_CUDA(dim == 3 ? gc::canonicalize<4>(d_simplices_in, n, num_vertices, B, st) : gc::canonicalize<3>(d_simplices_in, n, num_vertices, B, st));
  int bad = 0;
  GALE_CUDA(cudaMemcpyAsync(&bad, B.bad, 4, cudaMemcpyDeviceToHost, st));
  GALE_CUDA(cudaStreamSynchronize(st));  // the temporaries are released on return
  if (bad) { g_last_error = "a simplex names a vertex outside [0, num_vertices) or repeats one"; return GALE_ERR_DEGENERATE; }
  return GALE_OK;
}

// The same sort with its temporaries in g_canon_static_scratch instead of cudaMalloc'ed buffers (include/gale.h):
// for callers that cannot allocate. No cudaMalloc / cudaFree / allocating library call on this path. The first
// call on a device resolves the array's device address (canon_static_base) — do it before any stream capture.
int32_t gale_canonicalize_static(int32_t dim, int64_t num_simplices, int32_t num_vertices, const int32_t* d_simplices_in,
                                 int32_t* d_simplices_out, int32_t* d_perm_out, void* cuda_stream) {
  namespace gc = gale::canon;
  if ((dim != 2 && dim != 3) || num_simplices < 0 || num_vertices <= 0) return GALE_ERR_INVALID_ARG;
  if (num_simplices > kCanonStaticMaxN) {   // checked before any pointer or device is looked at
    g_last_error = "gale_canonicalize_static: num_simplices " + std::to_string((long long)num_simplices) +
                   " exceeds GALE_CANON_STATIC_MAX_SIMPLICES (" + std::to_string(kCanonStaticMaxN) +
                   "), the capacity of the library's built-in scratch; use gale_canonicalize";
    return GALE_ERR_WORKSPACE;
  }
  if (num_simplices > 0 && (!d_simplices_in || !d_simplices_out || d_simplices_in == d_simplices_out)) return GALE_ERR_INVALID_ARG;
  // one array per device shared by every call: nobody else may be sorting in it while this call's kernels run
  std::lock_guard<std::mutex> lock(g_canon_static_mutex);
  unsigned char* base = nullptr;
  int rc = canon_static_base(&base);
  if (rc != GALE_OK) return rc;
  if (num_simplices == 0) return GALE_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const long long n = num_simplices;
  gc::Buffers B;
  B.T[0] = d_simplices_out; B.T[1] = reinterpret_cast<int32_t*>(base + kCsT1);
  B.perm[0] = d_perm_out ? d_perm_out : reinterpret_cast<int32_t*>(base + kCsP0);
  B.perm[1] = reinterpret_cast<int32_t*>(base + kCsP1);
  B.counts = reinterpret_cast<int32_t*>(base + kCsCounts);   // every (digit, segment) counter is written by k_count
  B.scratch = reinterpret_cast<int32_t*>(base + kCsScan);    // every chunk sum is written by k_scan_sums
  B.bad = reinterpret_cast<int*>(base + kCsBad);             // only ever set by the kernels: must start at zero
  GALE_CUDA(cudaMemsetAsync(B.bad, 0, 4, st));
  GALE_CUDA(dim == 3 ? gc::canonicalize<4>(d_simplices_in, n, num_vertices, B, st) : gc::canonicalize<3>(d_simplices_in, n, num_vertices, B, st));
  int bad = 0;
  GALE_CUDA(cudaMemcpyAsync(&bad, B.bad, 4, cudaMemcpyDeviceToHost, st));
  GALE_CUDA(cudaStreamSynchronize(st));  // the scratch is free for the next call once this returns
  if (bad) { g_last_error = "a simplex names a vertex outside [0, num_vertices) or repeats one"; return GALE_ERR_DEGENERATE; }
  return GALE_OK;
}

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
  out->num_edges = m->nE;
  out->num_triangles = m->nF;
  out->kernel_variant = m->kernel;
  out->tune_dense_ms = m->tune_ms[0];
  out->tune_walk_ms = m->tune_ms[1];
  out->reserved = 0;
  return GALE_OK;
}

int32_t gale_mesh_tile(const gale_mesh_t* m, int32_t tile, gale_tile_view_t* out) {
  if (!m || !out || tile < 0 || tile >= m->plan->nTiles) return GALE_ERR_INVALID_ARG;
  const Plan& p = *m->plan;
  const TileDesc& t = p.tiles[size_t(tile)];
  out->v_lo = t.v_lo; out->nrows = t.nrows;
  out->t_lo = t.t_lo; out->num_internal = t.s_int;
  out->num_external = t.s_ext;
  out->num_lower_halo = t.nlo; out->num_local = t.nloc;
  out->cluster = int32_t(std::upper_bound(p.cl_tile_begin.begin(), p.cl_tile_begin.end(), tile) - p.cl_tile_begin.begin()) - 1;
  out->d_external = m->dm.tex + t.tex_off;
  out->d_local_to_global = m->dm.gid + t.gid_off;
  return GALE_OK;
}

int32_t gale_mesh_interval_array(const gale_mesh_t* m, const int32_t** d_first_simplex) {
  if (!m || !d_first_simplex) return GALE_ERR_INVALID_ARG;
  *d_first_simplex = m->dm.first_tet;
  return GALE_OK;
}

int32_t gale_mesh_edges(const gale_mesh_t* m, const int32_t** d_first, const int32_t** d_upper, int64_t* num_edges) {
  if (!m || !d_first || !d_upper || !num_edges) return GALE_ERR_INVALID_ARG;
  if (!m->sub.e_first) { g_last_error = "the edge list was not built (GALE_WITH_EDGES)"; return GALE_ERR_UNSUPPORTED; }
  *d_first = m->sub.e_first; *d_upper = m->sub.e_hi; *num_edges = m->nE;
  return GALE_OK;
}

int32_t gale_mesh_triangles(const gale_mesh_t* m, const int32_t** d_first, const int32_t** d_second_third, int64_t* num_triangles) {
  if (!m || !d_first || !d_second_third || !num_triangles) return GALE_ERR_INVALID_ARG;
  if (!m->sub.f_first) { g_last_error = "the triangle list was not built (GALE_WITH_FACETS)"; return GALE_ERR_UNSUPPORTED; }
  *d_first = m->sub.f_first; *d_second_third = reinterpret_cast<const int32_t*>(m->sub.f_bc); *num_triangles = m->nF;
  return GALE_OK;
}

int32_t gale_boundary_lookup(gale_mesh_t* m, int32_t relation, int64_t first_id, int64_t count, int32_t* d_out, void* cuda_stream) {
  namespace gs = gale::sub;
  if (!m || count < 0 || first_id < 0 || (count > 0 && !d_out)) return GALE_ERR_INVALID_ARG;
  if (relation != GALE_BND_FE && relation != GALE_BND_TE && relation != GALE_BND_TF) return GALE_ERR_INVALID_ARG;
  const bool need_e = relation != GALE_BND_TF, need_f = relation != GALE_BND_TE;
  if ((need_e && !m->sub.e_first) || (need_f && !m->sub.f_first)) {
    g_last_error = "the boundary relation needs the edge / triangle list (GALE_WITH_EDGES / GALE_WITH_FACETS at create)";
    return GALE_ERR_UNSUPPORTED;
  }
  const long long rows = relation == GALE_BND_FE ? m->nF : m->plan->nT;
  if (first_id + count > rows) return GALE_ERR_INVALID_ARG;
  if (count == 0) return GALE_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int W = gs::boundary_width(relation, m->D);
  const long long n = count * W;
  const unsigned blocks = (unsigned)((n + 255) / 256);
  const int32_t* T = m->dm.T;
  const int nV = m->plan->nV;
  if (relation == GALE_BND_FE) gs::k_boundary<gs::BND_FE, 4><<<blocks, 256, 0, st>>>(m->sub, T, nV, first_id, count, d_out);
  else if (relation == GALE_BND_TF) gs::k_boundary<gs::BND_TF, 4><<<blocks, 256, 0, st>>>(m->sub, T, nV, first_id, count, d_out);
  else if (m->D == 4) gs::k_boundary<gs::BND_TE, 4><<<blocks, 256, 0, st>>>(m->sub, T, nV, first_id, count, d_out);
  else gs::k_boundary<gs::BND_TE, 3><<<blocks, 256, 0, st>>>(m->sub, T, nV, first_id, count, d_out);
  GALE_CUDA(cudaGetLastError());
  return GALE_OK;
}

int32_t gale_cluster_batch_compute(gale_mesh_t* m, uint32_t relation_mask, const int32_t* h_cluster_ids,
                                   int32_t n_clusters, void* cuda_stream) {
  constexpr uint32_t kCobMask = GALE_REL_EF | GALE_REL_ET | GALE_REL_FT;
  if (!m || (relation_mask & ~uint32_t(GALE_REL_ALL | GALE_REL_VE | GALE_REL_VF | kCobMask)) || relation_mask == 0 || n_clusters < 0 ||
      (n_clusters > 0 && !h_cluster_ids))
    return GALE_ERR_INVALID_ARG;
  const uint32_t user_mask = relation_mask;
  if ((user_mask & GALE_REL_VE) && !m->sub.e_first) { g_last_error = "VE needs GALE_WITH_EDGES at create"; return GALE_ERR_UNSUPPORTED; }
  if ((user_mask & GALE_REL_VF) && !m->sub.f_first) { g_last_error = "VF needs GALE_WITH_FACETS at create"; return GALE_ERR_UNSUPPORTED; }
  // VE is a map over the VV rows, VF works on the VT rows: the batch kernel computes those too
  if ((user_mask & kCobMask) && !m->cob_ready) { g_last_error = "EF / ET / FT need GALE_WITH_COBOUNDARY at create"; return GALE_ERR_UNSUPPORTED; }
  // sources: VE, VF and EF are read off the VV rows, ET and FT off the VT rows (gale_sub.cuh)
  relation_mask = (user_mask & GALE_REL_ALL) | ((user_mask & (GALE_REL_VE | GALE_REL_VF | GALE_REL_EF)) ? GALE_REL_VV : 0u) |
                  ((user_mask & (GALE_REL_ET | GALE_REL_FT)) ? GALE_REL_VT : 0u);
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
  s.seq = seq; s.n = n_clusters; s.mask = user_mask | relation_mask; s.eff_mask = relation_mask;
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
    s.used.ve_idx = o; if (user_mask & GALE_REL_VE) o = up(o + size_t(s.vv_nnz) * 4, 16);
    s.vf_nnz = 0;
    if (user_mask & GALE_REL_VF) {
      for (int i = 0; i < n_clusters; ++i) s.vf_nnz += m->cl_cob[gale::sub::COB_VF][size_t(s.ids[i])];
      if (s.vf_nnz >= (1LL << 31) - 1) return GALE_ERR_INVALID_ARG;
      s.used.vf_off = o; o = up(o + size_t(s.rows + 1) * 4, 16);
      s.used.vf_idx = o; o = up(o + size_t(s.vf_nnz) * 4, 16);
    }
    if (user_mask & kCobMask) {
      s.e_row_begin.assign(size_t(n_clusters) + 1, 0);
      s.f_row_begin.assign(size_t(n_clusters) + 1, 0);
      for (int i = 0; i < n_clusters; ++i) {
        const int c = s.ids[size_t(i)];
        s.e_row_begin[size_t(i) + 1] = s.e_row_begin[size_t(i)] + (m->cl_e0[size_t(c) + 1] - m->cl_e0[size_t(c)]);
        s.f_row_begin[size_t(i) + 1] = s.f_row_begin[size_t(i)] + (m->cl_f0[size_t(c) + 1] - m->cl_f0[size_t(c)]);
      }
      const uint32_t bit[3] = {GALE_REL_ET, GALE_REL_FT, GALE_REL_EF};
      for (int k = 0; k < 3; ++k) {
        s.cob_nnz[k] = 0;
        if (!(user_mask & bit[k])) continue;
        for (int i = 0; i < n_clusters; ++i) s.cob_nnz[k] += m->cl_cob[k][size_t(s.ids[size_t(i)])];
        if (s.cob_nnz[k] >= (1LL << 31) - 1) return GALE_ERR_INVALID_ARG;
        const long long rows = k == gale::sub::COB_FT ? s.f_row_begin[size_t(n_clusters)] : s.e_row_begin[size_t(n_clusters)];
        s.used.cob_off[k] = o; o = up(o + size_t(rows + 1) * 4, 16);
        s.used.cob_idx[k] = o; o = up(o + size_t(s.cob_nnz[k]) * 4, 16);
      }
    }
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
  cfg.stage_t = (!walk && (p.flags & GALE_STAGE_FROM_T)) ? 1 : 0;
  if (cfg.stage_t && cfg.nloc == 0) cfg.nloc = p.cfg.nloc;  // the vertex table is needed for the mapping
  const gale::SmemLayout lay = layout_for(D, cfg);
  const gale::WalkLayout wlay = walk_layout_for(D, cfg);
#if GALE_CHECK_BOUNDS
  // negative control of the bounds-checked build: understate one capacity (the layout keeps its real
  // size) so that the kernel's checks must fire
  if (std::getenv("GALE_CHECK_SELFTEST") && cfg.vt_max > 8) cfg.vt_max -= 8;
#endif
  const int smem = walk ? wlay.total : lay.total;
  // everything the caller enqueued on its stream so far (e.g. the upload of the simplices) comes first
  cudaStream_t run = m->stream_ordered ? st : m->launch[seq % m->n_launch];
  if (!m->stream_ordered) {
    GALE_CUDA(cudaEventRecord(s.ev_submit, st));
    GALE_CUDA(cudaStreamWaitEvent(run, s.ev_submit, 0));
  }
  GALE_CUDA(cudaEventRecord(s.ev_start, run));
  // descriptor of the launch that covers the clusters [b, b + nb) of the batch (<= kMaxBatch per launch)
  auto fill_params = [&](int b, gale::BatchParams& P) -> int {
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
    return nb;
  };
  // First the VT / VV / TT rows of the WHOLE batch, launch by launch; only then the relations read off them. A row's
  // end is the next row's offset, and the next row may belong to the following launch: a VE / VF / EF / ET / FT launch
  // issued right after "its" batch-kernel launch would read the offset at the seam before anybody has written it.
  for (int b = 0; b < std::max(1, n_clusters); b += gale::kMaxBatch) {
    gale::BatchParams P{};
    const int nb = fill_params(b, P);
    const int grid = std::max(1, P.tile_prefix[nb]);
    if (walk) walk_kernel_for(D, p.w_NT, p.cfg.lb, relation_mask == GALE_REL_ALL)<<<grid, p.w_NT, smem, run>>>(m->dm, P, cfg, wlay, O);
    else kernel_for(D, p.NT, false, p.cfg.lb)<<<grid, p.NT, smem, run>>>(m->dm, P, cfg, lay, O);
    GALE_CUDA(cudaGetLastError());
  }
  for (int b = 0; (user_mask & (GALE_REL_VE | GALE_REL_VF | kCobMask)) && b < std::max(1, n_clusters); b += gale::kMaxBatch) {
    gale::BatchParams P{};
    const int nb = fill_params(b, P);
    const int grid = std::max(1, P.tile_prefix[nb]);
    if (nb > 0 && (user_mask & GALE_REL_VE)) {  // VE: a map over the VV rows just written (gale_sub.cuh)
      gale::sub::BatchRows B{};
      B.n_clusters = nb;
      for (int i = 0; i <= nb; ++i) B.row_base[i] = s.row_begin[b + i];
      for (int i = 0; i < nb; ++i) B.cluster[i] = s.ids[b + i];
      const int rows = B.row_base[nb] - B.row_base[0];
      if (rows > 0)
        gale::sub::k_ve<<<(rows + 127) / 128, 128, 0, run>>>(B, m->sub, O.vv_offsets, O.vv_indices,
                                                               reinterpret_cast<int32_t*>(s.dev + s.used.ve_idx));
      GALE_CUDA(cudaGetLastError());
    }
    if (user_mask & (GALE_REL_VF | kCobMask)) {  // VF / EF / ET / FT from the VT / VV rows just written
      namespace gs = gale::sub;
      const uint32_t bit[4] = {GALE_REL_ET, GALE_REL_FT, GALE_REL_EF, GALE_REL_VF};
      for (int k = 0; k < 4; ++k) {
        if (!(user_mask & bit[k])) continue;
        gs::CobParams V{};
        V.n_clusters = nb;
        V.uniform_tiles = P.uniform_tiles;
        if (k == gs::COB_VF) { V.total_rows = int(s.rows); V.total_nnz = int(s.vf_nnz); }
        else { V.total_rows = (k == gs::COB_FT ? s.f_row_begin : s.e_row_begin)[size_t(n_clusters)]; V.total_nnz = int(s.cob_nnz[k]); }
        long long base = 0;
        for (int i = 0; i < b; ++i) base += m->cl_cob[k][size_t(s.ids[size_t(i)])];
        for (int i = 0; i < nb; ++i) {
          V.tile_prefix[i + 1] = P.tile_prefix[i + 1];
          V.cluster[i] = P.cluster[i];
          V.src_row_base[i] = P.row_base[i];
          V.row_base[i] = k == gs::COB_VF ? P.row_base[i] : (k == gs::COB_FT ? s.f_row_begin : s.e_row_begin)[size_t(b + i)];
          V.nnz_base[i] = int(base);
          base += m->cl_cob[k][size_t(s.ids[size_t(b + i)])];
        }
        int32_t* ooff = reinterpret_cast<int32_t*>(s.dev + (k == gs::COB_VF ? s.used.vf_off : s.used.cob_off[k]));
        int32_t* oidx = reinterpret_cast<int32_t*>(s.dev + (k == gs::COB_VF ? s.used.vf_idx : s.used.cob_idx[k]));
        const bool from_vt = k == gs::COB_ET || k == gs::COB_FT;
        launch_star<false>(m, k, grid, V, from_vt ? O.vt_offsets : O.vv_offsets, from_vt ? O.vt_indices : O.vv_indices, ooff, oidx,
                           nullptr, nullptr, run);
        GALE_CUDA(cudaGetLastError());
      }
    }
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
  // A fired capacity guard is latched for the life of the handle (the flag is shared by all batches in flight, so
  // it cannot be pinned on one of them): the batch is popped all the same — its view must be released like any
  // other, its contents are unspecified — and this and every later pop report GALE_ERR_WORKSPACE. The queue keeps
  // moving, nobody spins on a slot that never frees.
  const int32_t guard = *static_cast<volatile int32_t*>(m->h_err);
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
  if (s.mask & GALE_REL_VE) out->ve_indices = reinterpret_cast<const int32_t*>(b + s.used.ve_idx);
  if (s.mask & (GALE_REL_EF | GALE_REL_ET | GALE_REL_FT)) {
    out->e_row_begin = s.e_row_begin.data();
    out->f_row_begin = s.f_row_begin.data();
    namespace gs = gale::sub;
    if (s.mask & GALE_REL_ET) { out->et_nnz = s.cob_nnz[gs::COB_ET]; out->et_offsets = reinterpret_cast<const int32_t*>(b + s.used.cob_off[gs::COB_ET]); out->et_indices = reinterpret_cast<const int32_t*>(b + s.used.cob_idx[gs::COB_ET]); }
    if (s.mask & GALE_REL_FT) { out->ft_nnz = s.cob_nnz[gs::COB_FT]; out->ft_offsets = reinterpret_cast<const int32_t*>(b + s.used.cob_off[gs::COB_FT]); out->ft_indices = reinterpret_cast<const int32_t*>(b + s.used.cob_idx[gs::COB_FT]); }
    if (s.mask & GALE_REL_EF) { out->ef_nnz = s.cob_nnz[gs::COB_EF]; out->ef_offsets = reinterpret_cast<const int32_t*>(b + s.used.cob_off[gs::COB_EF]); out->ef_indices = reinterpret_cast<const int32_t*>(b + s.used.cob_idx[gs::COB_EF]); }
  }
  if (s.mask & GALE_REL_VF) {
    out->vf_nnz = s.vf_nnz;
    out->vf_offsets = reinterpret_cast<const int32_t*>(b + s.used.vf_off);
    out->vf_indices = reinterpret_cast<const int32_t*>(b + s.used.vf_idx);
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
  if (guard != 0) {
    g_last_error = "device capacity guard fired: code " + std::to_string(guard);
    return GALE_ERR_WORKSPACE;
  }
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
