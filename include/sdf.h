/*
 * sdf.h -- C ABI of the B200-native CSC closest-point transform
 * (narrow-band signed distance + closest-triangle grids from a closed triangle soup).
 *
 * Method: Roosing, Strickson, Nikiforakis, "Fast Distance Fields for Fluid Dynamics
 * Mesh Generation on Graphics Hardware", arXiv:1903.00353.  Citations are lines of
 * /root/reference/PAPER.md ("PAPER.md:<line>") plus the section / equation.
 *
 *   problem statement      PAPER.md:45   (eq.1: f(x) = min distance to the surface, signed)
 *                          PAPER.md:63-77 (sec.2 pseudo-code: for each extrusion, for each cell
 *                                          inside, keep the min-magnitude distance)
 *   input                  PAPER.md:274-294 (sec.7: closed, consistently oriented STL triangle
 *                                          soup, vertices counter-clockwise from outside,
 *                                          arbitrary triangle order, duplicated vertices)
 *   grid / output          PAPER.md:384  (sec.10: row-major 1-D float array; coordinates
 *                                          recovered from the offset and the physical limits)
 *   band                   PAPER.md:392  (distance written only if smaller than a user maximum)
 *
 * Every function returns an int status (0 = SDF_OK); none throws, aborts or prints.
 * The library never falls back to a CPU implementation: without a CUDA device every
 * compute entry point returns SDF_ECUDA.
 * Threading: calls on one handle must not overlap, and neither may calls that create library-wide
 * state for the first time (the first sdf_create / sdf_compute of a process create the library's
 * side streams: vertex stage, sentinel fill); distinct handles on distinct streams are otherwise independent.
 * Debug / ablation switches (environment, read per call): SDF_AABB_MODE=1 (candidates = band-expanded
 * triangle boxes only), SDF_DISABLE=faces|wedges|cones (leave an extrusion class out: the parity harness must notice),
 * SDF_FILL_MODE=0..4, SDF_SCHEDULER=serial | dynamic[:N], SDF_RUFF=cone, SDF_NO_BINNING=1,
 * SDF_CREATE_FORK=0 (vertex stage on the caller's stream), SDF_SMOOTH_SIN=x (edges / vertices whose normals span less
 * than asin(x) get no wedge / cone of their own, their faces' prisms are widened instead; default 1/32, 0 = off), SDF_FILLINT_PLAIN=1 (interior fill without the blank map);
 * SDF_FILL_SM_SHARE=1..8 / SDF_FILL_CHUNK_LOG2=11..14 / SDF_FILL_ISSUERS=1..4 / SDF_FILL_DEPTH / SDF_SCRATCH_HINT=0 (sentinel-fill and scratch
 * ablations); SDF_ROW_CLIP=n (rows longer than n cells are clipped analytically before the walk; default 2), SDF_EVAL_CHUNK=n (warps per round in which faces, wedges and cones of a region are evaluated together; 0 = class after class);
 * see DESIGN.md.
 */
#ifndef PAPER_1903_00353_SDF_H
#define PAPER_1903_00353_SDF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    SDF_OK          = 0,
    SDF_EINVAL      = 1,  /* null pointer, ntri <= 0, h <= 0, band <= 0, bad dims, NaN/Inf input */
    SDF_ENOTCLOSED  = 2,  /* an undirected edge without exactly two incident triangles */
    SDF_EORIENT     = 3,  /* an edge traversed in the same direction by both triangles */
    SDF_EDEGENERATE = 4,  /* zero-area triangle or repeated vertex in a triangle */
    SDF_ENOMEM      = 5,  /* device (or host staging) allocation failed */
    SDF_ECUDA       = 6,  /* CUDA runtime error / no device; see sdf_last_cuda_error() */
    SDF_EIO         = 7,  /* file cannot be opened / read / written, or is not a valid STL file */
    SDF_ETOOBIG     = 8   /* sdf_fill_interior_static: the grid needs more scratch than the static array holds */
};

/* Opaque handle: device-resident feature tables of one mesh.  Owned by the library,
 * released by sdf_destroy. */
typedef struct sdf_mesh sdf_mesh;

/* Device-memory callbacks supplied by the caller (from Python: torch's caching
 * allocator).  `alloc` returns a DEVICE pointer usable on `stream` (NULL on failure);
 * `free` releases it.  Pass a NULL sdf_allocator* to let the library use the CUDA
 * stream-ordered pool (cudaMallocAsync). The struct is copied; `user` must stay valid
 * until sdf_destroy. */
typedef struct sdf_allocator {
    void *(*alloc)(size_t bytes, void *stream, void *user);
    void  (*free)(void *ptr, void *user);
    void  *user;
} sdf_allocator;

/* Counters of the feature builder and of the last sdf_compute (host values). */
typedef struct sdf_stats_t {
    int64_t F, V, E;                      /* triangles, welded vertices, undirected edges      */
    int64_t edges_convex, edges_concave, edges_flat;      /* PAPER.md:352 discriminant; knife   */
                                          /* edges (n1 = -n2) count as convex; edges_flat also  */
                                          /* counts the smooth edges absorbed by their faces    */
    int64_t verts_pos_only, verts_neg_only, verts_both, verts_skipped; /* cone sides emitted;  */
                                          /* skipped = smooth vertices absorbed by their faces  */
    int64_t verts_hemisphere;             /* "ruff" vertices: cos_cone <= 0 */
    int64_t weld_collisions;              /* reserved (always 0: the weld table probes, it has no runs) */
    /* last sdf_compute */
    int64_t polyhedra;                    /* extrusions with a non-empty clipped bounding volume */
    int64_t work_items;                   /* (polyhedron, grid row) items scan-converted        */
    int64_t pairs_tested;                 /* (cell, polyhedron) pairs a row loop looked at      */
    int64_t pairs_accepted;               /* of those: inside the polyhedron and d < band       */
    int64_t bricks_active, bricks_total;  /* 8x8x8-cell bricks holding packed scratch           */
    int64_t band_cells;                   /* populated output cells                             */
    int64_t fp64_rechecks;                /* cells whose band / sign decision was redone in fp64 */
                                          /* (cells without a certain sign from their candidate) */
    int64_t cdp_fallbacks;                /* SDF_SCHEDULER=dynamic only: child launches the device    */
                                          /* runtime refused (their volumes were walked serially)     */
} sdf_stats_t;

/*
 * sdf_create -- organise the unordered soup into features (sec.7: weld
 * identical vertices, pair the two half-edges of every edge
 * eq.8: angle-weighted pseudonormals; convex / concave /
 * flat / saddle classification) and build the band-independent part of every
 * characteristic polyhedron (eq.3-5, 344-364 sec.8).
 *
 *   tri_xyz   [ntri][3 vertices][x,y,z] fp32, counter-clockwise seen from outside
 *             (PAPER.md:278).  HOST pointer when on_device == 0 (copied with
 *             cudaMemcpyAsync), DEVICE pointer when on_device == 1.  Borrowed for the
 *             duration of the call only.  Vertices are identical iff their three fp32
 *             values are bit-identical (-0 == +0).
 *   ntri      1 .. 2^29
 *   a         device allocator, or NULL
 *   stream    cudaStream_t (0 = legacy default stream).  The call synchronises the stream
 *             once, before returning (validation flags and the counts of vertices, wedges and
 *             cones; the per-vertex tables are sized by V <= 3F/2 + 64, which every closed
 *             surface meets, so no count is needed mid-way).
 * The library works on a spatially ordered copy of the soup (fine Morton order); every
 * triangle id it reports is the caller's.  Vertex ids (sdf_get_table) and the order of the edge
 * records depend on the order in which thread blocks run; no value of the output grids does.
 * SDF_BUILDER=tile selects the tile-local builder (shared-memory weld / pairing per spatial tile;
 * bit-identical tables and grids, measured slower on a B200: an ablation).
 *   out       receives the handle on SDF_OK; set to NULL otherwise.
 * Errors: SDF_EINVAL, SDF_ENOTCLOSED, SDF_EORIENT, SDF_EDEGENERATE, SDF_ENOMEM, SDF_ECUDA.
 */
int sdf_create(const float *tri_xyz, int64_t ntri, int on_device,
               const sdf_allocator *a, void *stream, sdf_mesh **out);

/*
 * sdf_compute -- clip every characteristic polyhedron to the band and the grid
 * (PAPER.md:344-364), scan-convert it row by row (sec.5, replacing the
 * schedulers of PAPER.md:366-380), evaluate the exact feature distance for every cell
 * inside and min-combine, then sign every populated cell --
 * from the polarity of the winning extrusion where that is certain, else
 * from the pseudonormal of its closest feature -- and write both grids.
 *
 *   origin    HOST pointer to 3 floats: position of sample (0,0,0).  Sample (i,j,k) sits at
 *             origin + (i,j,k)*h (cell centres).
 *   h         grid spacing > 0;  nx,ny,nz: 1 .. 32767 each;  band in length units,
 *             0 < band <= 250 * h (the paper's bands are 5 .. 62 cells).
 *   dist_out  DEVICE, caller-owned, nx*ny*nz floats, linear index ((int64)k*ny + j)*nx + i
 *             (x fastest).  Signed distance, negative inside, written iff
 *             |d| < band; +INFINITY elsewhere.  Every element is
 *             overwritten.
 *   tri_out   DEVICE, caller-owned, nx*ny*nz int32: index (in the caller's soup order) of
 *             the closest triangle, -1 outside the band.  Where several triangles are
 *             equally close (closest point on a shared edge / vertex) the lowest index.
 *   stream    cudaStream_t.  Work is enqueued on it; the call synchronises it once
 *             mid-way (active-brick total) and leaves the final kernels enqueued.  The
 *             dense sentinel write runs on a library-owned stream that is forked from and
 *             joined back into `stream` with events (stream-ordered for the caller).
 * May be called repeatedly on one handle with different grids / bands.
 * Errors: SDF_EINVAL, SDF_ENOMEM, SDF_ECUDA.
 */
int sdf_compute(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz,
                float band, float *dist_out, int32_t *tri_out, void *stream);

/*
 * sdf_transform -- one pass of the whole hot path A0-A8 on one mesh and one grid: sdf_create
 * followed by sdf_compute, with identical results (bit for bit), arguments, layouts and error
 * behaviour; every argument is checked before any work is enqueued.  Knowing the grid before the
 * feature construction lets the dense sentinel write of both grids (A8a:
 * +INFINITY / -1 outside the band), which depends on nothing but the output
 * pointers, start earlier: environment SDF_PREFILL_AT = 1 (before A0), 2 (before the edge table),
 * 3 (before edge pairing), 4 (default: behind the last feature kernel, under the host crossing),
 * 5 (after the crossing, where sdf_compute forks it).  On a B200 the starts 1-3 LOSE: the feature
 * kernels and the fill are bound by the same memory pipe and take the sum of their times whatever
 * the fill's rate, so they are an ablation.  What the single call does gain: the
 * brick marking and its prefix sum (A6a) run inside the feature construction and their total
 * returns with the validation flags -- ONE stream synchronisation for the whole call against two
 * for the two calls (SDF_HOIST_BRICKS=0 switches that off).
 *
 *   tri_xyz, ntri, on_device, a      as for sdf_create
 *   origin, h, nx, ny, nz, band      as for sdf_compute
 *   dist_out, tri_out                DEVICE, caller-owned, as for sdf_compute; overwritten entirely
 *   stream                           cudaStream_t; synchronised once (flags, counts and the brick total together)
 *   out                              receives the handle (for sdf_stats, further sdf_compute calls ...) on
 *                                    SDF_OK; NULL otherwise, and then the output grids hold unspecified values
 *                                    (the fill has been waited for: nothing is left in flight).
 * Errors: those of sdf_create and sdf_compute; arguments are checked before any work is enqueued.
 */
int sdf_transform(const float *tri_xyz, int64_t ntri, int on_device, const sdf_allocator *a,
                  const float origin[3], float h, int nx, int ny, int nz, float band,
                  float *dist_out, int32_t *tri_out, void *stream, sdf_mesh **out);

/*
 * sdf_zslab / sdf_compute_zslab -- the paper's multi-card outlook (a domain
 * "distributed across multiple cards"): the grid is cut into `parts` slabs of whole z-slices and
 * every process computes one of them from the complete feature tables of its own handle.  No cell
 * of a slab needs anything from another slab (every polyhedron that reaches it is evaluated
 * locally), so there is no halo and no exchange: the slabs are independent sdf_compute calls.
 *
 * sdf_zslab (host only, no CUDA): slab `part` of `parts` of a grid of nz slices is
 * [*k0, *k0 + *nk); boundaries fall on multiples of 8 slices (the brick height), the slabs are
 * disjoint, ordered, cover [0, nz), and differ by at most 8 slices; *nk may be 0 when
 * parts > ceil(nz / 8).  Errors: SDF_EINVAL (nz < 1, parts < 1, part outside [0, parts), NULL).
 *
 * sdf_compute_zslab: sdf_compute on the grid (nx, ny, *nk) whose sample (0,0,0) sits at
 * origin + (0, 0, k0 * h), the z component evaluated in double and rounded once to float (that
 * float IS the slab's origin: sample k of the slab sits at fmaf(k, h, origin_z'), which equals
 * the whole grid's fmaf(k0 + k, h, origin_z) whenever both are exact, e.g. for power-of-two h,
 * and differs from it by at most one rounding otherwise).  dist_out / tri_out: DEVICE,
 * nx*ny*(*nk) elements, slab-local linear index.  k0_out / nk_out (HOST, may be NULL) receive
 * the range.  An empty slab returns SDF_OK without touching the outputs.
 * Errors: those of sdf_zslab and sdf_compute.
 */
int sdf_zslab(int nz, int part, int parts, int *k0, int *nk);
int sdf_compute_zslab(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz,
                      float band, int part, int parts, float *dist_out, int32_t *tri_out,
                      void *stream, int *k0_out, int *nk_out);

/*
 * sdf_compute_host -- same as sdf_compute but dist_out / tri_out are HOST buffers
 * (pinned memory recommended): device grids are taken from the allocator, computed,
 * copied back with cudaMemcpyAsync and the stream is synchronised before returning.
 */
int sdf_compute_host(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz,
                     float band, float *dist_out_host, int32_t *tri_out_host, void *stream);

/*
 * sdf_compute_sparse / sdf_compute_sparse_host -- the same narrow band in band-sparse storage: only the 8x8x8-cell
 * bricks the band can reach are stored (at C4: 43,350 of 2,097,152 bricks, 178 MB instead of 8.6 GB), the way level-set
 * codes keep a band (PAPER.md:392 writes a distance only inside the band; PAPER.md:493 names the dense grid as the limit
 * of the method's reach).  Identical values to sdf_compute, cell for cell (tests/test_gpu_sparse.py); no dense grid is
 * allocated, filled or copied.
 *
 *   origin, h, nx, ny, nz, band   as for sdf_compute
 *   brick_cap     capacity of the three outputs, in bricks (0 is allowed: the call then only counts)
 *   brick_ids     int32 [brick_cap]: linear index (bz * nby + by) * nbx + bx of each stored brick, ascending, with
 *                 nbx = ceil(nx / 8) etc.; brick (bx,by,bz) holds the cells 8*bx .. 8*bx+7 (clipped to the grid) etc.
 *   dist_bricks   float [brick_cap][512]: cell (i,j,k) of its brick at [(k & 7) * 64 + (j & 7) * 8 + (i & 7)]; signed
 *                 distance, +INFINITY where |d| >= band or the cell lies outside the grid; 16-byte aligned
 *   tri_bricks    int32 [brick_cap][512]: closest triangle id, -1 where dist is +INFINITY; 16-byte aligned
 *   nbricks_out   HOST: the number of bricks the band reaches.  If it exceeds brick_cap nothing is written and the call
 *                 returns SDF_ENOMEM: call again with at least that capacity (the count costs A6a only, not the evaluation)
 *   stream        cudaStream_t; synchronised once mid-way (the brick count), like sdf_compute
 * sdf_compute_sparse: outputs in DEVICE memory, left enqueued on `stream`.  sdf_compute_sparse_host: outputs in HOST
 * memory (pinned recommended): staged on the device through the allocator, copied back (only *nbricks_out bricks) and
 * the stream synchronised before returning.
 * Errors: SDF_EINVAL, SDF_ENOMEM (also: brick_cap too small), SDF_ECUDA.
 */
int sdf_compute_sparse(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz, float band, int64_t brick_cap,
                       int32_t *brick_ids, float *dist_bricks, int32_t *tri_bricks, int64_t *nbricks_out, void *stream);
int sdf_compute_sparse_host(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz, float band,
                            int64_t brick_cap, int32_t *brick_ids_host, float *dist_bricks_host, int32_t *tri_bricks_host,
                            int64_t *nbricks_out, void *stream);

/*
 * sdf_closest_points -- the closest point transform proper: for every cell whose
 * closest-triangle id (as written by sdf_compute on the same grid) is >= 0, the point of that
 * triangle nearest to the cell centre; +INFINITY in all three components elsewhere.
 *
 *   origin, h, nx, ny, nz   the grid sdf_compute was called with
 *   tri_in    DEVICE, nx*ny*nz int32, the tri_out of sdf_compute
 *   cp_out    DEVICE, caller-owned, nx*ny*nz*3 floats, [cell][x,y,z], cells in the order of dist_out
 *   stream    cudaStream_t; one kernel is enqueued, nothing is synchronised
 * Errors: SDF_EINVAL, SDF_ECUDA.
 */
int sdf_closest_points(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz,
                       const int32_t *tri_in, float *cp_out, void *stream);

/*
 * sdf_fill_interior -- PAPER.md:493 (sec.11.3): the narrow band leaves "a secondary zero crossing
 * between the negative limit of the SDF and the interior of the surface beyond the maximum
 * distance", fixed "by sweeping along each of the coordinate axes and filling in unset values in
 * the interior of the geometry".  Operates in place on a dist grid written by sdf_compute: for the
 * axes x, y, z in turn every grid line is walked forward and then backward; a walk keeps the sign
 * of the last set (finite) cell, and an unset (+INFINITY) cell met while that sign is negative is
 * set to -band.  Cells outside the solid stay +INFINITY; the band itself and tri_out are not touched.
 *
 *   dist      DEVICE, nx*ny*nz floats, layout of sdf_compute (x fastest)
 *   band      the band width sdf_compute was called with (the value written is -band)
 *   stream    cudaStream_t; the three sweeps are enqueued on it, nothing is synchronised
 * Scratch: nx*ny*nz/128 bytes (one bit per 32-cell row segment, twice) from the device's default
 * memory pool with cudaMallocAsync / cudaFreeAsync on `stream`; the pool's release threshold is
 * raised to twice that size plus 64 MiB if it is lower (the one process-wide setting the library
 * changes; the pool reserves in chunks and would otherwise hand them back at every synchronisation).
 * Errors: SDF_EINVAL, SDF_ENOMEM, SDF_ECUDA.
 */
int sdf_fill_interior(float *dist, int nx, int ny, int nz, float band, void *stream);

/*
 * sdf_fill_interior_static -- sdf_fill_interior for callers that must not allocate: code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same arguments, same result cell for cell.
 * The scratch (the two blank maps, nx*ny*nz/128 bytes for nx a multiple of 1024) is a static device array of
 * 8 MiB inside the library -- every GPU that loads the library holds it until the process exits -- so:
 *   - a grid with ny * nz * ceil(nx / 1024) > 2^20 (more than 1024^3 cells at nx = 1024) is refused: SDF_ETOOBIG,
 *     nothing is launched;
 *   - the call performs no cudaMalloc, cudaFree, cudaMallocAsync or memory-pool call; it enqueues three kernels on
 *     `stream` and returns (the first call on a device also looks the array's address up: cudaGetSymbolAddress);
 *   - all calls share the one array: two calls that may overlap on the GPU (streams without an order between them,
 *     concurrent host threads) race on it and their results are undefined.  Calls ordered on one stream are safe;
 *     the array needs no clearing between them.
 * Errors: SDF_EINVAL, SDF_ETOOBIG, SDF_ECUDA.
 */
int sdf_fill_interior_static(float *dist, int nx, int ny, int nz, float band, void *stream);

/*
 * STL and grid files (host code; "takes as input a stereolithography (STL) file and
 * outputs a file that lists the SDF values in a 3D grid"; ASCII facet layout PAPER.md:278-288).
 *
 * sdf_read_stl   binary or ASCII (detected), -> HOST array [ntri][3 vertices][xyz] allocated by the
 *                library (release with sdf_free_host), in file order, ready for sdf_create with
 *                on_device = 0.  The facet normals of the file are ignored: orientation is the
 *                counter-clockwise vertex order.
 * sdf_write_stl  ascii != 0: ASCII with 9 significant digits (fp32 round-trips), else binary.
 * sdf_write_grid the library's own layout (the paper gives none): "SDFGRID1", int32 nx, ny, nz,
 *                has_tri, float origin[3], h, band, nx*ny*nz floats (x fastest), then, if tri_host is
 *                not NULL, nx*ny*nz int32.  dist_host / tri_host are HOST buffers.
 * Errors: SDF_EINVAL, SDF_EIO, SDF_ENOMEM.
 */
int  sdf_read_stl(const char *path, float **tri_xyz_out, int64_t *ntri_out);
void sdf_free_host(void *p);
int  sdf_write_stl(const char *path, const float *tri_xyz, int64_t ntri, int ascii);
int  sdf_write_grid(const char *path, const float *dist_host, const int32_t *tri_host,
                    const float origin[3], float h, int nx, int ny, int nz, float band);

/* Counters (host struct filled from the handle; synchronises `the last stream used` if a
 * compute is still in flight). */
int sdf_stats(sdf_mesh *m, sdf_stats_t *out);

/*
 * sdf_get_table -- copy one internal feature table to HOST memory (tests / inspection).
 *   which: one of SDF_TABLE_*; dst: host buffer of `bytes` bytes, which must equal the
 *   table size exactly (SDF_EINVAL otherwise).  Synchronous.
 */
enum {
    SDF_TABLE_CORNER_VID   = 0,  /* int32 [3F]   corner -> welded vertex id                      */
    SDF_TABLE_HALFEDGE_ADJ = 1,  /* int32 [3F]   half-edge 3t+k (corner k -> k+1) -> its opposite */
    SDF_TABLE_FACE_NORMAL  = 2,  /* float [F][3] unit face normals                               */
    SDF_TABLE_VERTEX_REC   = 3,  /* 32 B  [V]    {float pos[3], axis[3], cos_cone; int32 info}; info bit0 / bit1: cone on
                                    the + / - side of the axis, bit2: hemisphere (ruff), bit3: smooth vertex (no cone
                                    of its own: its region is covered by the widened prisms of its faces)           */
    SDF_TABLE_EDGE_REC     = 4,  /* 64 B  [edges_convex + edges_concave]  {float a[3], b[3], n1[3], n2[3]; int32 tri, cls,
                                    pad[2]}: one record per edge that has a wedge, in no particular order; flat and
                                    smooth edges (counted in edges_flat) have none                                   */
    SDF_TABLE_VERTEX_MINTRI= 5   /* int32 [V]    lowest incident triangle id                     */
};
int sdf_get_table(sdf_mesh *m, int which, void *dst, size_t bytes);

/*
 * Stage timing (measurement support).  sdf_enable_timing(1) makes every
 * later sdf_create / sdf_compute record CUDA events around its stages ON THE STREAM IT WAS
 * GIVEN (no extra synchronisation); sdf_enable_timing(2) records only the two events around the
 * dense sentinel write (SDF_T_FILL, the kernel the roofline is quoted on), so that a timed step
 * carries next to no instrumentation; 0 switches it off.  sdf_get_timings synchronises that stream and returns
 * the durations, in milliseconds, of the stages of the handle's sdf_create and of its last
 * sdf_compute.  ms: HOST array of SDF_T_COUNT floats (n must equal SDF_T_COUNT); a stage
 * that did not run reports 0.
 */
enum {
    SDF_T_INGEST_WELD = 0,  /* A0+A1: spatial binning, gather/canonicalise, weld table, vertex ids */
    SDF_T_EDGES       = 1,  /* A2+A3: triangle geometry, half-edge table, pairing, edge classes   */
    SDF_T_VERTICES    = 2,  /* A3+A4: pseudonormals, cone angles, vertex classes (library-owned
                               second stream, concurrent with the pairing part of stage 1)       */
    SDF_T_CLIP_SCAN   = 3,  /* A6a: brick marks, prefix sum, brick table, the host crossing       */
    SDF_T_CLEAR       = 4,  /* scratch bricks reset to "empty"                                    */
    SDF_T_EVALUATE    = 5,  /* A5-A7: clip, scan-convert, distances, packed atomicMin             */
    SDF_T_EMIT        = 6,  /* A8b: sign pass over the active bricks, written into both grids     */
    SDF_T_FILL        = 7,  /* A8a: dense sentinel fill of both grids (library-owned side stream,
                               concurrent with stage 5)                                         */
    SDF_T_COUNT       = 8
};
int sdf_enable_timing(int on);
int sdf_get_timings(sdf_mesh *m, float *ms, int n);

/*
 * sdf_measure_fp32_peak -- measurement support for the FP32 leg of the roofline (BASELINE.json north_star: "the
 * candidate cell x feature distance evaluations at FP32 peak"): runs a register-resident FMA loop
 * (16 independent chains per thread, 2048 threads per SM) six times on `stream`, synchronises, and returns the best
 * rate in TFLOP/s (2 flop per FMA) in *tflops_out (HOST); *sm_count_out (HOST, may be NULL) receives the SM count.
 * Nominal on a B200: 148 SMs x 128 FMA lanes x 2 x 1.965 GHz = 74.4 TFLOP/s.
 * Errors: SDF_EINVAL, SDF_ENOMEM, SDF_ECUDA.
 */
int sdf_measure_fp32_peak(double *tflops_out, int *sm_count_out, void *stream);

/* Number of CUDA kernels this library has launched in this process so far. */
int64_t sdf_launch_count(void);

/* Release the handle and all its device memory (NULL is a no-op). */
void sdf_destroy(sdf_mesh *m);

/* Static string for a status code. */
const char *sdf_strerror(int status);

/* cudaError_t value of the last failing CUDA call seen by this library (0 if none). */
int sdf_last_cuda_error(void);

/* Library version, for the symbol / load test. */
int sdf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PAPER_1903_00353_SDF_H */
