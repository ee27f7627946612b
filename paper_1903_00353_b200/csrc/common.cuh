// common.cuh -- shared declarations of the CUDA path (sm_100a).
// Shares nothing with oracle/ (the CPU oracle is test infrastructure).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/sdf.h"

typedef unsigned int u32;
typedef unsigned long long u64;

// ---------------------------------------------------------------------------------------
// error handling: every CUDA call goes through CK(); the first failure is remembered
// ---------------------------------------------------------------------------------------
extern int g_last_cuda_error;
extern int g_timing;                 // sdf_enable_timing
extern long long g_launch_count;     // kernels launched by this library (sdf_launch_count)
#define KL (++g_launch_count)        // written in front of every <<< >>> launch
#define CK(call)                                                   \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) {                                  \
            g_last_cuda_error = (int)e__;                          \
            (void)cudaGetLastError();                              \
            return (e__ == cudaErrorMemoryAllocation) ? SDF_ENOMEM : SDF_ECUDA; \
        }                                                          \
    } while (0)
#define CKS(expr)                                                  \
    do {                                                           \
        int s__ = (expr);                                          \
        if (s__ != SDF_OK) return s__;                             \
    } while (0)

// error bits raised by device code (sdf_mesh::d_flags[0])
enum { ERRB_NONFINITE = 1, ERRB_NOTCLOSED = 2, ERRB_ORIENT = 4, ERRB_DEGENERATE = 8 };

// device counters (sdf_mesh::d_ctr), 64-bit each
enum {
    CTR_V = 0, CTR_ELIVE, CTR_E_CONVEX, CTR_E_CONCAVE, CTR_E_FLAT,      // ELIVE: edge records written (wedges that exist)
    CTR_V_POS, CTR_V_NEG, CTR_V_BOTH, CTR_V_SKIP, CTR_V_HEMI, CTR_NCONE,   // NCONE: entries of the cone list
    CTR_POLY, CTR_ITEMS, CTR_BRICKS, CTR_TESTED, CTR_ACCEPTED, CTR_BAND, CTR_RECHECK,
    CTR_BIG, CTR_CDP_FALLBACK,   // big-polyhedron list length (fetch cursors: CTR_BIGCUR); refused child launches (cdp.cu)
    CTR_COUNT = 24,
    // statistics that every warp adds to are spread over CTR_SLOTS lines of 8 counters
    // (same-address atomics serialise in L2); sdf_stats sums the slots
    CTR_SPREAD = CTR_COUNT, CTR_SLOTS = 64,
    CTR_BIGCUR = CTR_SPREAD + CTR_SLOTS * 8,     // evaluate_big_kernel: one fetch cursor per row slice
    CTR_TOTAL = CTR_BIGCUR + 8
};
enum { SP_POLY = 0, SP_TESTED, SP_ACCEPTED, SP_ROWS, SP_BAND, SP_RECHECK };

// ---------------------------------------------------------------------------------------
// feature tables (HBM layout)
// ---------------------------------------------------------------------------------------
// Band-independent part of an edge wedge: end points in the direction the
// half-edge is traversed in triangle t0 (normal n1), n2 = normal of the opposite triangle.
struct __align__(16) EdgeRec {
    float a[3], b[3], n1[3], n2[3];
    int tri;     // min(t0, t1): the id written for cells closest to this edge
    int cls;     // +1 convex, -1 concave, 0 flat (no wedge), 2 knife (faces folded back: whole cylinder)
    int pad[2];
};
static_assert(sizeof(EdgeRec) == 64, "EdgeRec must be 64 B");

// Band-independent part of a vertex cone: apex, unit pseudonormal axis
// (eq.8), cosine of the half angle (eq.9), info bits.
struct __align__(16) VertexRec {
    float pos[3], axis[3];
    float cos_cone;
    int info;    // bit0: emit +axis side, bit1: emit -axis side, bit2: hemisphere (ruff),
                 // bit3: smooth vertex, no cone of its own: absorbed by the margins of its faces
};
static_assert(sizeof(VertexRec) == 32, "VertexRec must be 32 B");

// Smooth features: an edge whose two face normals, or a vertex whose cone of normals,
// spans less than asin(SMOOTH_SIN) gets no polyhedron of its own.  Its characteristic region (the wedge of PAPER.md:352,
// the cone of eq.9) lies within reach * sin(angle) of the side planes of every incident face's prism -- a
// point p + r d with p on the face and d at angle a from the face normal projects r sin(a) away from p -- so each
// incident face widens its prism sideways by that much and evaluates the clamped point-triangle distance there, which is
// the distance to the edge / vertex.  (At C4 the dihedral angles are ~3e-3: 5.9 M wedges and 2-4 M cones, 99 % of them
// without a single cell centre inside, become a 0.6 % wider face prism.)
#define SMOOTH_SIN_DEFAULT 0.03125f
// sine of twice the half angle of a vertex cone from its (already widened) stored cosine, rounded up
#define VSM_SCALE 8192.0f           // byte code of a smooth vertex' margin sine (SMOOTH_SIN_DEFAULT * VSM_SCALE = 256)
__device__ __forceinline__ float cone_sin2(float c) {
    if (!(c > 0.9f)) return INFINITY;
    return 2.0f * c * sqrtf(fmaxf(0.0f, 1.0f - c * c)) * 1.00001f + 1e-7f;
}

// Band- and grid-dependent bounding volume of one polyhedron in cell indices, clipped to the grid
// (PAPER.md:348, 364, 370), and the number of grid rows (j,k) it covers.  Lives in registers only.
struct PolyHdr {
    short i0, i1, j0, j1, k0, k1;
    u32 rows;
    float msin;                      // face slabs: sine of the sideways margin for the smooth features it absorbs
};

#define BIG_ROWS 256u                // ... when it has more rows than this
#define BIG_NI 32                    // ... or rows at least this long

#define BRICK 8                      // scratch bricks are 8x8x8 cells
#define BRICK_CELLS 512
#define PACK_EMPTY 0xFFFFFFFFFFFFFFFFull

struct GridParams {
    float ox, oy, oz, h, inv_h;
    double dox, doy, doz, dh;       // same values promoted (fp64 re-check paths)
    int nx, ny, nz;
    int nbx, nby, nbz;              // bricks per axis
    float band, eps, guard, rb;     // rb = band + guard + eps : reach of every polyhedron
    double dband;
    int big_rows, big_ni;           // polyhedra with more rows / longer rows go to evaluate_big_kernel
    int plain_cpt;                  // debug: closest points with the dense one-pass kernel only
    int serial_loop;                // ablation: the paper's thread-per-extrusion serial loop
    int cdp, cdp_serial_below;      // ablation: the paper's dynamic-parallelism scheduler (cdp.cu)
    int aabb_mode;                  // debug: candidates = band-expanded triangle AABBs only
    int disable;                    // debug (harness self-test): extrusion classes left out, bit0 face slabs, bit1 edge wedges, bit2 vertex cones
    int vec4;                       // 1: nx % 4 == 0 and outputs 16-B aligned -> 128-bit stores
    int fill_mode;                  // 0: TMA fill on the side stream (default); debug: 1 plain stores on the
                                    // side stream, 2 TMA fill on the main stream before the emit, 3 ... first,
                                    // 4 forked after the mid-way host crossing
    int fill_prio;                  // side stream at the highest priority
    int fill_ctas;                  // TMA fill: CTAs launched per SM (one per SM survives)
    float tiny_abs;                 // an fp32 distance at or below this has no reliable sign: 2 ulp of the largest |coordinate| of the grid
    int row_clip;                   // rows longer than this many cells are clipped analytically before they are walked
    int eval_chunk;                 // warps per class-interleaving round of evaluate_small_kernel (0: plain order)
    int fill_depth, fill_issuers;   // TMA fill: chunk pairs in flight per issuing lane, issuing lanes per SM
    int scratch_hint;               // L2 evict-last hint on the scratch atomics (default on)
    int fill_chunk_log2;            // TMA fill: log2 of the bytes per bulk copy (11..14)
    int fill_sm_share;              // TMA fill: SMs out of every 8 that stream (8 = all; fewer = throttled, ablation)
};

// ---------------------------------------------------------------------------------------
// handle
// ---------------------------------------------------------------------------------------
struct sdf_mesh {
    sdf_allocator alloc;     // copied; alloc.alloc == nullptr -> cudaMallocAsync
    int64_t F, E, V;
    // device memory comes in a few slabs carved into tables (one allocator call each: the
    // caller's allocator may be a slow host callback)
    void *slab_f;            // every persistent feature table (per-vertex ones sized by V <= 3F/2 + 64) + counters
    void *slab_ws; size_t slab_ws_cap;     // per-compute workspace (bytes), grown on demand
    // feature tables (device, views into the slabs)
    float *soup;             // [F][9] canonicalised copy of the input
    float *fn;               // [F][3] unit face normals
    int *perm;               // [F] internal triangle index -> the caller's id (spatial binning)
    int *inv_perm;           // [F] the caller's id -> internal index
    int *cvid;               // [3F]
    int *adj;                // [3F]
    int *vmint;              // [V]
    VertexRec *vrec;         // [V]
    EdgeRec *erec;           // [E] capacity; Elive records written: the wedges that exist (not flat, not absorbed)
    float *fsm;              // [F] face margin factor: max sine of the angle between the normals over the smooth EDGES the
                             //     face absorbs (its smooth vertices are looked up by the evaluation: evaluate.cuh
                             //     face_margin_sin); the prism is widened sideways by reach * that sine
    unsigned char *vsm;      // [V] smooth vertices: ceil(8192 * sine of the full cone angle) (1..255), 0 = not smooth.  What the
                             //     evaluation looks up per face corner: a table small enough to stay in L2
    u32 *cone_list;          // [2V] capacity; NC entries (vertex id << 1 | side): the vertex cones that exist
    int64_t Elive, NC;
    u64 *d_ctr;              // [CTR_COUNT]
    int *d_flags;            // [4]
    // persistent per-compute workspace (grown on demand)
    u64 *scan_ws;
    unsigned char *brick_flag;
    int *brick_table;
    int *brick_list;                       // scratch slot -> brick index
    u32 *big_list;                         // polyhedra of evaluate_big_kernel
    u32 *fill_state;                       // fill_tma_kernel: batch cursor + per-SM claims
    u32 *cp_state;                         // same, for the +inf fill of sdf_closest_points (own allocation)
    u64 *scratch;  size_t scratch_cap;     // bricks * 512 packed values
    u64 h_ctr[CTR_COUNT];
    cudaEvent_t ev[SDF_T_COUNT][2];   // stage begin / end events (created on first use)
    bool ev_set[SDF_T_COUNT];
    int64_t last_bricks_total;
    cudaStream_t last_stream;
    cudaStream_t side;                // library-owned stream of the sentinel fill (A8a)
    cudaEvent_t ev_fork, ev_join;
    int ev_dev1;                      // 1 + device the handle's pooled events belong to (0: none taken yet)
    cudaEvent_t ev_bjoin;             // join of the brick stream (hoisted A6a beside the edge and vertex stages)
    // sdf_transform: sentinel fill still to be started at stage boundary pre_at of build_features (0 = none pending)
    const GridParams *pre_g; float *pre_dist; int *pre_tri; int pre_at;
    // sdf_transform: A6a (brick marks + scan) still to be run by build_features / already run for the next run_compute
    const GridParams *hoist_g; bool bricks_ready;
    GridParams *hoist_g_dev;          // device copy of the grid for kernels of sdf_create that mark bricks (sdf_transform)
    cudaEvent_t ev_ffork, ev_fjoin;   // fork / join of the sentinel fill (ev_fork / ev_join: the vertex stream)
};

// carve 256-byte aligned tables out of one slab; with base == nullptr it only adds up sizes
struct Carver {
    char *base; size_t off;
    explicit Carver(void *b) : base((char *)b), off(0) {}
    template <typename T> T *take(size_t n) {
        off = (off + 255) & ~(size_t)255;
        T *p = base ? (T *)(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

// the library's fork / join events come from a process-wide pool (creating and destroying five per handle was a tenth of
// the host time of a small sdf_transform); thread-safe; an event goes back when its handle is destroyed
struct sdf_mesh;
int ev_get(sdf_mesh *m, cudaEvent_t *e);          // no-op if *e is set already
void ev_put(sdf_mesh *m, cudaEvent_t *e);

// allocation through the handle's allocator
int dev_alloc(const sdf_allocator *a, void **p, size_t bytes, cudaStream_t st);
void dev_free(const sdf_allocator *a, void *p, cudaStream_t st);

// stage timing: record the begin (which = 0) / end (which = 1) event of a stage on st
void stage_mark(sdf_mesh *m, int stage, int which, cudaStream_t st);

// stages (features.cu / compute.cu)
int build_features(sdf_mesh *m, const float *tri, int on_device, cudaStream_t st);
// band-sparse output of run_compute (sdf_compute_sparse): bricks instead of dense grids
struct SparseOut { int64_t cap; int *ids; float *dist; int *tri; int64_t count; };
int run_compute(sdf_mesh *m, const GridParams &g, float *dist, int *tri, cudaStream_t st, bool prefilled = false,
                SparseOut *sp = nullptr);
int start_prefill(sdf_mesh *m, const GridParams &g, float *dist, int *tri, cudaStream_t st);
int maybe_prefill(sdf_mesh *m, int point, cudaStream_t st);
int maybe_alloc_brick_ws(sdf_mesh *m, cudaStream_t st);
int maybe_begin_bricks(sdf_mesh *m, cudaStream_t st, const GridParams **g_dev, unsigned char **flag);
int maybe_prepare_bricks(sdf_mesh *m, cudaStream_t st, cudaStream_t vs, bool marked);
int run_closest_points(sdf_mesh *m, const GridParams &g, const int *tri, float *cp, cudaStream_t st);
