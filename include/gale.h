/* gale.h — C ABI of the B200-native GALE relation hot path.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, arXiv 2507.15230):
 *   GALE's "worker producers" (PAPER.md:160 §4.2, :226-280 §4.6, Alg. 1 :232-250): for a batch of
 *   mesh segments ("clusters"), the coboundary relation VT and the adjacency relations VV and TT
 *   (§2.2, Table 1 :53-58), delivered to the consumer side through a bounded queue of
 *   pre-allocated buffers (PAPER.md:158 leader producer; :208 "pre-allocates sufficient GPU memory").
 *   Readings of everything the paper leaves open are listed in DESIGN.md §Readings.
 *
 * Input contract ("canonical mesh"): D = dim+1 vertex ids per simplex, int32;
 *   (C1) each row strictly ascending, (C2) rows strictly ascending lexicographically,
 *   (C3) ids in [0, num_vertices), (C4) every facet has at most two cofaces.
 *   Cluster c owns the vertices [o[c], o[c+1]) (I_V, Alg. 1 line 3 :243) and the
 *   *internal* simplices {t : o[c] <= T[t][0] < o[c+1]}, a contiguous id range by C2.
 *
 * Output per cluster, canonical sorted CSR, all stored ids GLOBAL:
 *   VT rows v = o[c]..o[c+1]-1 : ascending ids of the simplices containing v (internal + external);
 *   VV rows v                  : ascending ids of the distinct vertices u != v sharing a simplex with v;
 *   TT rows t in I_T[c]        : D entries; entry k = the simplex sharing the facet opposite the k-th
 *                                smallest vertex of t, or -1 on the boundary.
 *
 * No CPU fallback exists: without an sm_100 CUDA device every compute entry returns
 * GALE_ERR_UNSUPPORTED / GALE_ERR_CUDA. No exception crosses this boundary.
 * Thread-safety: one producer thread (compute) + one consumer thread (pop/release) per handle.
 */
#ifndef GALE_H_
#define GALE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gale_mesh gale_mesh_t; /* opaque; owned by the library, freed by gale_destroy */
typedef struct gale_plan gale_plan_t; /* opaque result of the initialization analysis, see gale_plan_create */

enum {
  GALE_REL_VT = 1, GALE_REL_VV = 2, GALE_REL_TT = 4,
  GALE_REL_ALL = 7,  /* the three relations of the hot path                                           */
  GALE_REL_VE = 8,   /* vertex -> incident edges; needs GALE_WITH_EDGES at create; also delivers VV   */
  GALE_REL_VF = 16,  /* vertex -> incident triangles (tetrahedral meshes); needs GALE_WITH_FACETS; also
                        delivers VV (its source)                                                     */
  /* the coboundary relations of edges and triangles (Table 1; MS complex :309), tetrahedral
     meshes, need GALE_WITH_COBOUNDARY; rows = the edges / triangles internal to the requested clusters
     (those whose lowest vertex belongs to the cluster), in id order; EF also delivers VV,
     ET and FT also deliver VT (the rows they are read off)                                            */
  GALE_REL_EF = 32,  /* edge -> triangles                                                             */
  GALE_REL_ET = 64,  /* edge -> simplices                                                             */
  GALE_REL_FT = 128  /* triangle -> simplices (one or two)                                            */
};

enum {
  GALE_OK = 0,
  GALE_ERR_INVALID_ARG = -1,   /* null pointer, bad dim, relation_mask == 0, ...                      */
  GALE_ERR_NOT_CANONICAL = -2, /* C1-C3 violated (checked when GALE_VALIDATE is set)                  */
  GALE_ERR_DEGENERATE = -3,    /* gale_canonicalize: a simplex repeats a vertex or names one out of range */
  GALE_ERR_NONMANIFOLD = -4,   /* C4 violated (checked when GALE_VALIDATE_MANIFOLD is set)            */
  GALE_ERR_BAD_CLUSTER = -5,   /* cluster id out of range, or n_clusters > max_batch_clusters         */
  GALE_ERR_WOULD_BLOCK = -6,   /* every queue slot is un-released (compute), or timeout (pop)         */
  GALE_ERR_EMPTY = -7,         /* pop with nothing in flight                                          */
  GALE_ERR_WORKSPACE = -8,     /* workspace too small / misaligned, or a device capacity guard fired  */
  GALE_ERR_CUDA = -9,          /* a CUDA call failed; see gale_last_error()                           */
  GALE_ERR_UNSUPPORTED = -10   /* no sm_100 device, or a vertex star too large for shared memory      */
};

enum {
  GALE_VALIDATE = 1u,          /* check C1-C3 and the cluster offsets at create (one pass)            */
  GALE_VALIDATE_MANIFOLD = 2u, /* also check C4 (facet pass, slower)                                  */
  GALE_KERNEL_DENSE = 8u,      /* force the dense kernel (one thread per staged simplex)              */
  GALE_KERNEL_WALK = 16u,      /* force the walk kernel (two threads per tile vertex); UNSUPPORTED if
                                  its capacity limits do not admit the mesh. Neither flag: create times
                                  both on a sample batch and keeps the faster (gale_mesh_info tells)   */
  GALE_WITH_EDGES = 64u,       /* initialization also builds the sorted edge list E and its interval array
                                  I_E (generated "only when the edge or triangle information
                                  is explicitly needed"); enables GALE_REL_VE                              */
  GALE_WITH_FACETS = 128u,     /* ... and the sorted triangle list F with I_F; enables GALE_REL_VF (dim = 3)  */
  GALE_WITH_COBOUNDARY = 256u, /* with GALE_WITH_EDGES | GALE_WITH_FACETS (dim = 3): also size EF / ET / FT and reserve
                                  room for them in the result slots; enables GALE_REL_EF / _ET / _FT          */
  GALE_STAGE_FROM_T = 32u,     /* stage the rows of T and T_ex themselves and derive the tile-local ids in the
                                  kernel instead of reading the create-time re-encoding; only the dense kernel
                                  can, so the flag selects it (as GALE_KERNEL_DENSE does; with GALE_KERNEL_WALK:
                                  GALE_ERR_INVALID_ARG); slower, kept for the A/B in DESIGN.md              */
  GALE_STREAM_ORDERED = 4u     /* run every batch kernel on the cuda_stream passed to compute itself
                                  (plain stream order: work the caller enqueues afterwards runs after
                                  the batch) instead of on the library's two overlapping launch streams */
};

typedef struct {
  int32_t dim;                      /* 3 = tetrahedra, 2 = triangles                                  */
  int32_t num_vertices;
  int64_t num_simplices;            /* every simplex id must fit int32                                */
  const int32_t *d_simplices;       /* DEVICE, [num_simplices*(dim+1)], canonical, 16-byte aligned;
                                       caller-owned, must outlive the handle, never written by the
                                       library; its CONTENTS must not change while the handle lives
                                       (see gale_plan_create)                                         */
  int32_t num_clusters;
  const int32_t *h_cluster_offsets; /* HOST, [num_clusters+1], I_V: 0 = o[0] <= ... <= o[nC] = nV;
                                       read during create only                                       */
  int32_t max_batch_clusters;       /* largest n_clusters of one compute call (e.g. 64)               */
  int32_t queue_depth;              /* > 0: that many pinned HOST result slots, results are copied
                                       D2H on a library-owned side stream;
                                       0: results stay in a ring of device slots (benchmark mode)     */
  int32_t device_ring;              /* queue_depth == 0 only: number of device slots (0 = default 4)   */
  int32_t tile_vertices;            /* vertices per thread-block tile, <= 256 (0 = automatic: 32 for
                                       tets — 24 when 32-vertex tiles would need more than 28 KB of shared
                                       memory per block — and 64 for triangles; create may reduce any request that
                                       exceeds a kernel limit — gale_mesh_info reports the value used) */
  void *d_workspace;                /* DEVICE, caller-owned (e.g. a torch tensor), 256-byte aligned,
                                       must outlive the handle                                       */
  size_t workspace_bytes;
  uint32_t flags;                   /* GALE_VALIDATE | GALE_VALIDATE_MANIFOLD | GALE_STREAM_ORDERED |
                                       GALE_KERNEL_DENSE / GALE_KERNEL_WALK                           */
} gale_mesh_desc_t;

/* One finished batch. cluster_ids and *_row_begin are HOST arrays owned by the library; offsets and
 * indices live in the slot: pinned HOST memory when queue_depth > 0, DEVICE memory when 0
 * (on_device tells which). Everything stays valid until gale_queue_release, in both modes: a slot is
 * reused only after its view has been released (the paper's pre-allocated relation buffers).
 * Rows of the i-th requested cluster are [row_begin[i], row_begin[i+1]); offsets are batch-relative
 * (offsets[0] = 0, non-decreasing, offsets[rows] = nnz). TT rows have constant length dim+1. */
typedef struct {
  int64_t sequence;              /* submission order, from 0                                         */
  int32_t n_clusters;
  uint32_t relation_mask;
  int32_t dim;
  int32_t on_device;
  const int32_t *cluster_ids;    /* HOST [n_clusters], as passed to compute                          */
  const int32_t *vt_row_begin;   /* HOST [n_clusters+1] (also the VV row partition)                  */
  const int32_t *tt_row_begin;   /* HOST [n_clusters+1]                                              */
  int64_t vt_rows, vt_nnz;
  const int32_t *vt_offsets;     /* [vt_rows+1] or NULL when VT was not requested                    */
  const int32_t *vt_indices;     /* [vt_nnz]                                                         */
  int64_t vv_rows, vv_nnz;
  const int32_t *vv_offsets;     /* [vv_rows+1] or NULL                                              */
  const int32_t *vv_indices;     /* [vv_nnz]                                                         */
  int64_t tt_rows;
  const int32_t *tt_indices;     /* [tt_rows*(dim+1)] or NULL                                        */
  float kernel_ms;               /* CUDA-event time of this batch's kernel, start to end; it includes
                                    the time the GPU was shared with an overlapping neighbour batch  */
  int32_t slot;                  /* internal: pass the view back unchanged to gale_queue_release     */
  /* stages of a request as the paper times them: data preparation, kernel (above),
   * transfer back, and the wait of the consumer; "data integration" (:210) does not exist here        */
  float prep_ms;                 /* host time inside gale_cluster_batch_compute (batch set-up + launch) */
  float d2h_ms;                  /* queue_depth > 0: end of kernel -> copy landed in the pinned slot
                                    (includes waiting behind earlier copies on the side stream); else 0 */
  float queue_ms;                /* host time from the end of compute to the return of this pop         */
  int32_t reserved;
  /* edges / triangles. VE has the rows and offsets of VV: ve_indices[i] is the id of the
   * edge between the row's vertex and vv_indices[i]. Edge / triangle ids = positions in the sorted lists E / F */
  const int32_t *ve_indices;     /* [vv_nnz] or NULL                                                   */
  int64_t vf_nnz;
  const int32_t *vf_offsets;     /* [vt_row_begin[n_clusters]+1] (one row per vertex, like VT / VV) or NULL */
  const int32_t *vf_indices;     /* [vf_nnz]                                                           */
  /* EF / ET / FT: rows of the i-th requested cluster are [e_row_begin[i], e_row_begin[i+1]) (edges) resp.
   * f_row_begin (triangles); the first row of cluster c is edge I_E[o[c]] resp. triangle I_F[o[c]]     */
  const int32_t *e_row_begin;    /* HOST [n_clusters+1] or NULL                                        */
  const int32_t *f_row_begin;    /* HOST [n_clusters+1] or NULL                                        */
  int64_t ef_nnz, et_nnz, ft_nnz;
  const int32_t *ef_offsets, *ef_indices;   /* [edge rows + 1], [ef_nnz]: triangle ids                 */
  const int32_t *et_offsets, *et_indices;   /* [edge rows + 1], [et_nnz]: simplex ids                  */
  const int32_t *ft_offsets, *ft_indices;   /* [triangle rows + 1], [ft_nnz]: simplex ids              */
} gale_batch_view_t;

/* Init statistics ("Initialization"), for reporting. */
typedef struct {
  int32_t tile_vertices, num_tiles;
  int64_t num_external_refs;     /* total length of the per-tile T_ex lists                          */
  int64_t vt_nnz, vv_nnz;        /* whole-mesh totals                                                */
  int32_t smem_bytes;            /* dynamic shared memory per thread block of the batch kernel       */
  int32_t max_staged;            /* largest per-tile staged simplex count                            */
  size_t slot_bytes;             /* bytes of one result slot                                         */
  size_t workspace_used;
  double create_ms;
  int32_t local_id_bytes;        /* width of the tile-local vertex ids in the staged lists: 1 when every
                                    tile has at most 255 local vertices (tile + halo), else 2           */
  int32_t block_threads;         /* threads per block of the batch kernel                            */
  size_t index_bytes;            /* bytes of the device-resident index built by the initialization
                                    (I_T, T_ex, tile tables; the rest of workspace_used is result slots) */
  int64_t num_edges, num_triangles; /* sizes of E / F when built (GALE_WITH_EDGES / GALE_WITH_FACETS), else 0 */
  int32_t kernel_variant;        /* 0 = dense kernel, 1 = walk kernel (chosen at create, or forced)     */
  float tune_dense_ms, tune_walk_ms; /* sample-batch times behind that choice (0 = not timed)           */
  int32_t reserved;
} gale_mesh_info_t;

/* Canonical form of a simplex list, on the device (the form gale_plan_create expects,
 * DESIGN.md §2 reading 2): every row ascending, rows in ascending lexicographic order — the order in which
 * the simplices internal to a segment (lowest vertex in the segment) are one contiguous range,
 * which is what the interval array I_T of the paper's initialization records.
 *   d_simplices_in   DEVICE int32[num_simplices * (dim + 1)], vertex ids in any order inside a row, rows in any
 *                    order; valid in stream order on cuda_stream; not modified
 *   d_simplices_out  DEVICE int32[num_simplices * (dim + 1)], caller-owned, must not alias the input
 *   d_perm_out       DEVICE int32[num_simplices] or NULL: output row i is input row d_perm_out[i]. The sort is
 *                    stable (equal rows keep their input order), so the permutation is unique
 * dim is 2 or 3; num_vertices bounds the ids (it fixes the number of radix passes). Temporary device memory
 * (one more copy of the rows and of the permutation, 1 KB of counters per 2,048 rows) is the library's and is
 * released before return; the call synchronises cuda_stream. Errors: GALE_ERR_INVALID_ARG (NULL / aliased
 * arrays, bad dim or sizes), GALE_ERR_DEGENERATE (a row repeats a vertex or names one outside
 * [0, num_vertices); the output is then unspecified), GALE_ERR_CUDA, GALE_ERR_UNSUPPORTED (no sm_100 device). */
int32_t gale_canonicalize(int32_t dim, int64_t num_simplices, int32_t num_vertices, const int32_t *d_simplices_in,
                          int32_t *d_simplices_out, int32_t *d_perm_out, void *cuda_stream);

/* gale_canonicalize for callers that must not allocate device memory. Same operation, same arguments, same
 * results and error codes as gale_canonicalize above — but this entry
 * never calls cudaMalloc / cudaFree or any library routine that allocates.
 *
 * Who needs it: an analysis that runs in situ next to a simulation which has handed all of the GPU's memory to
 * its own pool (a cudaMalloc from a guest library fails there with out-of-memory although the pool could spare
 * the room), and a service loop that cannot afford the device-wide synchronisation cudaMalloc / cudaFree imply.
 * Such callers bring their input and output arrays; what the radix sort needs besides them (the second copy of
 * the rows, two permutation buffers, the per-segment digit counters, the error flag) lives in ONE array that is
 * part of the library image itself:
 *   - it is GALE_CANON_STATIC_SCRATCH_BYTES (about 25 MiB) of device memory on EVERY GPU on which this library's
 *     kernels get loaded, taken when the library's code is loaded there and held until the process exits, whether
 *     or not this entry is ever called;
 *   - it bounds the problem: num_simplices > GALE_CANON_STATIC_MAX_SIMPLICES returns GALE_ERR_WORKSPACE (with a
 *     text in gale_last_error) before anything is launched; larger lists need gale_canonicalize;
 *   - every call on a device uses the same array. Two calls whose kernels could overlap on the GPU would corrupt
 *     each other's sort, so the library holds a process-wide lock from entry until cuda_stream has drained; do not
 *     call it from a callback that this very stream waits on. The array keeps whatever the last call left in it;
 *     the one word that has to start at zero (the error flag) is cleared by every call, all other parts are
 *     fully overwritten before they are read.
 * The first call on each device (with that device current) looks up the device address of the array and checks the
 * device's compute capability; make that first call at set-up time, outside any CUDA stream capture. The call
 * synchronises cuda_stream, like gale_canonicalize. */
#define GALE_CANON_STATIC_MAX_SIMPLICES (1 << 20)
#define GALE_CANON_STATIC_SCRATCH_BYTES                                                                             \
  ((size_t)GALE_CANON_STATIC_MAX_SIMPLICES * (16 + 4 + 4) /* rows, two permutations */                              \
   + (size_t)(GALE_CANON_STATIC_MAX_SIMPLICES / 2048) * 1024 /* digit counters */ + 512 /* scan sums, error flag */)
int32_t gale_canonicalize_static(int32_t dim, int64_t num_simplices, int32_t num_vertices, const int32_t *d_simplices_in,
                                 int32_t *d_simplices_out, int32_t *d_perm_out, void *cuda_stream);

/* Initialization analysis ("Initialization": I_T, the external lists T_ex, interval
 * arrays): reads the simplices from the DEVICE array desc->d_simplices — they must be valid in stream
 * order on cuda_stream — validates them and builds the index with device kernels (csrc/gale_init.cuh) in
 * memory the library allocates and owns until the plan is consumed; the simplices never leave the GPU
 * (exception: GALE_VALIDATE_MANIFOLD checks C4 on a host copy). This is the expensive part of creating a
 * handle (about a third of a second for a 100 M-tet mesh on a warm context; the first CUDA call of a process
 * adds its context and module load); d_workspace / workspace_bytes of the descriptor are ignored. *out is
 * owned by the caller until it is passed to gale_mesh_create_planned or gale_plan_destroy.
 * The index is a digest of the VALUES of d_simplices at this moment: from here until gale_destroy the
 * array's contents are frozen. The batch kernels read the index, not the array (only the cross-cluster TT
 * look-ups and gale_boundary_lookup read it), so overwriting it with another mesh is not detected and
 * yields results of the old mesh, or garbage; a new mesh needs a new plan and a new handle. */
int32_t gale_plan_create(const gale_mesh_desc_t *desc, void *cuda_stream, gale_plan_t **out);

/* Exact device workspace (index + result slots) a handle built from this plan needs. Cheap. */
int32_t gale_plan_workspace_bytes(const gale_plan_t *plan, size_t *out_bytes);

int32_t gale_plan_destroy(gale_plan_t *plan);

/* Builds the handle from a plan: uploads the index into d_workspace (DEVICE, caller-owned, 256-byte
 * aligned, >= gale_plan_workspace_bytes, must outlive the handle) on cuda_stream, synchronised on return.
 * The plan is consumed (emptied) on every outcome; destroy it afterwards. */
int32_t gale_mesh_create_planned(gale_plan_t *plan, void *d_workspace, size_t workspace_bytes, void *cuda_stream,
                                 gale_mesh_t **out);

/* Convenience: gale_plan_create + gale_plan_workspace_bytes + gale_plan_destroy. NOT cheap: it runs the
 * whole analysis (see gale_plan_create; d_simplices must be valid on cuda_stream) and throws it away.
 * Callers that go on to create a handle should use the plan calls and pay for the analysis once. */
int32_t gale_mesh_workspace_bytes(const gale_mesh_desc_t *desc, void *cuda_stream, size_t *out_bytes);

/* Convenience: gale_plan_create + gale_mesh_create_planned with desc->d_workspace / workspace_bytes
 * (PAPER.md:178-180). Work is enqueued on cuda_stream (a cudaStream_t, 0 = default stream) and
 * finished (synchronised) on return. *out is set on GALE_OK only. */
int32_t gale_mesh_create(const gale_mesh_desc_t *desc, void *cuda_stream, gale_mesh_t **out);

/* Statistics of the initialization (Table 4 :393-397 reports its time), for reporting. */
int32_t gale_mesh_info(const gale_mesh_t *mesh, gale_mesh_info_t *out);

/* What the initialization built for one tile (the interval array I_T and the external list
 * T_ex of a segment; a tile is this library's segment). For inspection and tests. The
 * DEVICE pointers point into the workspace and stay valid as long as the handle. */
typedef struct {
  int32_t v_lo, nrows;            /* the tile's vertices [v_lo, v_lo + nrows)                          */
  int32_t t_lo, num_internal;     /* I_T: its internal simplices [t_lo, t_lo + num_internal)           */
  int32_t num_external;           /* length of its T_ex list                                           */
  int32_t num_lower_halo, num_local; /* vertices sharing a simplex with the tile, below it / tile + halo */
  int32_t cluster;                /* the cluster the tile belongs to                                   */
  const int32_t *d_external;      /* DEVICE [num_external] ascending simplex ids (T_ex)                */
  const int32_t *d_local_to_global; /* DEVICE [num_local] ascending vertex ids: halo below, tile, halo above */
} gale_tile_view_t;

/* tile in [0, gale_mesh_info().num_tiles); tiles are numbered cluster by cluster, ascending v_lo. */
int32_t gale_mesh_tile(const gale_mesh_t *mesh, int32_t tile, gale_tile_view_t *out);

/* DEVICE pointer to the interval array I_T per vertex, [num_vertices + 1]: entry v = first simplex whose
 * lowest vertex is >= v, so the internal simplices of any vertex range [lo, hi) are
 * [I[lo], I[hi]). */
int32_t gale_mesh_interval_array(const gale_mesh_t *mesh, const int32_t **d_first_simplex);

/* Boundary relations FE, TE, TF (Table 1 :53-58) by the look-up of PAPER.md:186-192: "retrieve the
 * boundary vertices ... locate edge indices through the edge list E with limiting the search range by the edge
 * interval array I_E" — one interval-bounded binary search per face, on the device, for a range of rows:
 *   GALE_BND_FE  rows = triangles [first_id, first_id + count) of F, 3 edge ids each          (dim 3, E and F built)
 *   GALE_BND_TE  rows = simplices of T, 6 edge ids each (3 for a triangle mesh)               (E built)
 *   GALE_BND_TF  rows = simplices of T, 4 triangle ids each                                   (dim 3, F built)
 * Entry j of a row is the j-th vertex combination in lexicographic order ((v0,v1), (v0,v2), .. — the order of the
 * paper's example FE(f5) = (v0,v3), (v0,v4), (v3,v4)). The remaining boundary relations are the lists themselves
 * (EV = gale_mesh_edges, FV = gale_mesh_triangles, TV = the caller's simplices).
 *   d_out  DEVICE int32[count * width], caller-owned; written in stream order on cuda_stream (asynchronous)
 * Errors: GALE_ERR_INVALID_ARG (relation, range), GALE_ERR_UNSUPPORTED (list not built), GALE_ERR_CUDA. */
enum { GALE_BND_FE = 1, GALE_BND_TE = 2, GALE_BND_TF = 3 };
int32_t gale_boundary_lookup(gale_mesh_t *mesh, int32_t relation, int64_t first_id, int64_t count, int32_t *d_out,
                             void *cuda_stream);

/* The sorted edge list E with its interval array, when built: the edges whose lowest vertex
 * is a are the ids [d_first[a], d_first[a+1]) and d_upper[id] is their other vertex (ascending). DEVICE
 * memory owned by the library, valid as long as the handle. GALE_ERR_UNSUPPORTED when not built. */
int32_t gale_mesh_edges(const gale_mesh_t *mesh, const int32_t **d_first, const int32_t **d_upper, int64_t *num_edges);
/* Likewise the triangle list F: d_second_third holds two ids per triangle. */
int32_t gale_mesh_triangles(const gale_mesh_t *mesh, const int32_t **d_first, const int32_t **d_second_third,
                            int64_t *num_triangles);

/* Producer side: enqueue the relation kernels for the clusters
 * h_cluster_ids[0..n) (HOST array, copied before return; duplicates are legal) and, when
 * queue_depth > 0, the D2H copy into a pinned slot on the library's side stream.
 * Stream semantics, default: the kernels run on library-owned streams (consecutive batches alternate
 * between two of them so that the draining tail of one launch overlaps the next), ORDERED AFTER
 * everything already enqueued on cuda_stream at the time of the call — e.g. an upload of the simplices.
 * Work the caller enqueues on cuda_stream afterwards is NOT ordered after the batch: completion is
 * observed through gale_queue_pop only, and the simplices / workspace must not be modified or freed
 * before the batches using them have been popped (gale_destroy drains them).
 * With GALE_STREAM_ORDERED in desc->flags the kernels run on cuda_stream itself: plain stream order,
 * later work on that stream sees the device slot complete (no overlap between consecutive batches).
 * Asynchronous w.r.t. the host. Returns GALE_ERR_WOULD_BLOCK when all slots are un-released.
 * The results describe the mesh as it was at create: the simplex array must still hold the same values. */
int32_t gale_cluster_batch_compute(gale_mesh_t *mesh, uint32_t relation_mask, const int32_t *h_cluster_ids,
                                   int32_t n_clusters, void *cuda_stream);

/* Consumer side (PAPER.md:158 "signals the consumer", :194: the consumer blocks until its relation is
 * there): wait (up to timeout_ms; < 0 = forever) for the oldest submitted batch and describe it in *out. Batches pop in submission order. GALE_ERR_EMPTY if nothing is in flight,
 * GALE_ERR_WOULD_BLOCK on timeout. GALE_ERR_WORKSPACE: a device-side capacity guard fired in this or another batch
 * of the handle; the batch IS popped and *out describes it (contents unspecified) — release it like any other view.
 * The condition is latched: every later pop of the handle reports it the same way, so a consumer loop must treat
 * any status other than GALE_OK / GALE_ERR_WOULD_BLOCK / GALE_ERR_EMPTY as fatal, drain and destroy the handle. */
int32_t gale_queue_pop(gale_mesh_t *mesh, gale_batch_view_t *out, int32_t timeout_ms);

/* Give a popped slot back to the queue (the relation buffers are pre-allocated and reused,
 * never freed per request). Mandatory in BOTH modes: a slot whose view was popped but not released keeps
 * gale_cluster_batch_compute at GALE_ERR_WOULD_BLOCK once the ring wraps around to it.
 * GALE_ERR_INVALID_ARG for a view that is not the popped, un-released view of its slot. */
int32_t gale_queue_release(gale_mesh_t *mesh, const gale_batch_view_t *view);

/* End of the producers' life (the producers serve requests until the consumers are done):
 * drains in-flight work, frees pinned memory, streams and events. The workspace and the simplex
 * array stay the caller's. */
int32_t gale_destroy(gale_mesh_t *mesh);

const char *gale_status_string(int32_t status);
/* Text of the last CUDA failure seen by this thread's calls ("" if none). */
const char *gale_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GALE_H_ */
