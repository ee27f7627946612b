// evaluate.cuh -- device-side pieces shared by the evaluation kernels of compute.cu and by the
// dynamic-parallelism ablation of cdp.cu (a translation unit of its own: it is the only one built
// as relocatable device code): vector helpers, the exact point-triangle routine, the polyhedron
// index space and its bounding volumes (A5), the packed atomicMin (A7,
// PAPER.md:374, 392) and the paper's per-thread serial walk of one bounding volume.
#pragma once
#include "common.cuh"
#include <math.h>

// ---------------------------------------------------------------------------------------
// small vector helpers (fp32 / fp64)
// ---------------------------------------------------------------------------------------
template <typename T> struct V3 { T x, y, z; };
typedef V3<float> f3;
template <typename T> __device__ __forceinline__ V3<T> mk(T x, T y, T z) { V3<T> r; r.x = x; r.y = y; r.z = z; return r; }
template <typename T> __device__ __forceinline__ V3<T> operator-(V3<T> a, V3<T> b) { return mk<T>(a.x - b.x, a.y - b.y, a.z - b.z); }
template <typename T> __device__ __forceinline__ V3<T> operator+(V3<T> a, V3<T> b) { return mk<T>(a.x + b.x, a.y + b.y, a.z + b.z); }
template <typename T> __device__ __forceinline__ V3<T> operator*(T s, V3<T> a) { return mk<T>(s * a.x, s * a.y, s * a.z); }
template <typename T> __device__ __forceinline__ T dot(V3<T> a, V3<T> b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <typename T> __device__ __forceinline__ V3<T> cross(V3<T> a, V3<T> b) {
    return mk<T>(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}
__device__ __forceinline__ f3 ld3(const float *p) { return mk<float>(p[0], p[1], p[2]); }
// dot product with a fixed association (no compiler contraction): the canonical form of every
// distance that reaches the output, so a value does not depend on the kernel that produced it
__device__ __forceinline__ float dot_rn(f3 a, f3 b) {
    return __fmaf_rn(a.z, b.z, __fmaf_rn(a.y, b.y, __fmul_rn(a.x, b.x)));
}
__device__ __forceinline__ V3<double> ld3d(const float *p) { return mk<double>((double)p[0], (double)p[1], (double)p[2]); }

enum { RG_FACE = 0, RG_E0 = 1, RG_E1 = 2, RG_E2 = 3, RG_V0 = 4, RG_V1 = 5, RG_V2 = 6 };

// Closest point of triangle (0, e0, ec) to r (everything relative to corner a), unit normal n.
// Formulation: if the projection falls inside all three in-plane edge half-planes the closest
// point is the projection (distance |n.r|, "n . pc"); otherwise it is on one of
// the edges whose half-plane is violated: clamped point-segment distances (PAPER.md:392
// "distance to a line", "distance between two points").  Returns the distance, the region
// and q = closest point relative to a.
template <typename T>
__device__ __forceinline__ T tri_closest(V3<T> r, V3<T> e0, V3<T> ec, V3<T> n, int &region, V3<T> &q) {
    V3<T> e1 = ec - e0;
    T s0 = dot(cross(n, e0), r);
    T s1 = dot(cross(n, e1), r - e0);
    T s2 = -dot(cross(n, ec), r - ec);
    if (s0 >= (T)0 && s1 >= (T)0 && s2 >= (T)0) {
        T dn = dot(n, r);
        q = r - dn * n;
        region = RG_FACE;
        return fabs(dn);
    }
    T best = (T)INFINITY;
    region = RG_V0;
    q = mk<T>(0, 0, 0);
    if (s0 < (T)0) {                     // segment a -> b
        T t = dot(r, e0) / dot(e0, e0);
        t = t < (T)0 ? (T)0 : (t > (T)1 ? (T)1 : t);
        V3<T> c = t * e0, d = r - c;
        T d2 = dot(d, d);
        if (d2 < best) { best = d2; q = c; region = t <= (T)0 ? RG_V0 : (t >= (T)1 ? RG_V1 : RG_E0); }
    }
    if (s1 < (T)0) {                     // segment b -> c
        V3<T> rb = r - e0;
        T t = dot(rb, e1) / dot(e1, e1);
        t = t < (T)0 ? (T)0 : (t > (T)1 ? (T)1 : t);
        V3<T> c = e0 + t * e1, d = r - c;
        T d2 = dot(d, d);
        if (d2 < best) { best = d2; q = c; region = t <= (T)0 ? RG_V1 : (t >= (T)1 ? RG_V2 : RG_E1); }
    }
    if (s2 < (T)0) {                     // segment c -> a
        V3<T> rc = r - ec;
        T t = -dot(rc, ec) / dot(ec, ec);
        t = t < (T)0 ? (T)0 : (t > (T)1 ? (T)1 : t);
        V3<T> c = ((T)1 - t) * ec, d = r - c;
        T d2 = dot(d, d);
        if (d2 < best) { best = d2; q = c; region = t <= (T)0 ? RG_V2 : (t >= (T)1 ? RG_V0 : RG_E2); }
    }
    return sqrt(best);
}

// ---------------------------------------------------------------------------------------
// A5 + A6a: per polyhedron, bounding volume in cell indices clipped to the grid, row count,
// and the bricks it may touch.  Polyhedron index space:
//   [0,F) face slabs | [F,F+E) edge wedges | [F+E, F+E+2V) vertex cones (+axis, -axis)
// ---------------------------------------------------------------------------------------
struct MeshView {
    const float *soup, *fn, *fsm;
    const unsigned char *vsm;
    const EdgeRec *erec;
    const VertexRec *vrec;
    const u32 *cone_list;
    const int *vmint, *cvid, *adj;
    const int *perm, *inv_perm;     // internal triangle index <-> the caller's id
    int F, E, V;                    // E = edge records (live wedges), not 3F/2
    int NC;                         // entries of cone_list
    int64_t P;                      // F + E + NC
};


// Cell-index range of [mn, mx] along one axis, clipped to the grid.  fp32: the index estimate
// (x - o) / h carries a rounding error below 32767 * 2^-22 < 8e-3 cells, covered by the slack
// (a superset only costs candidate cells; every candidate gets the exact tests).
#define CELL_SLACK 1e-2f
__device__ __forceinline__ void cell_range(float mn, float mx, float o, float inv_h, int n, int &lo, int &hi) {
    float l = ceilf((mn - o) * inv_h - CELL_SLACK), u = floorf((mx - o) * inv_h + CELL_SLACK);
    l = fminf(fmaxf(l, 0.0f), (float)n);
    u = fmaxf(fminf(u, (float)(n - 1)), -1.0f);
    lo = (int)l; hi = (int)u;
}

// A6a: the 8x8x8-cell bricks that can receive a distance.  Every polyhedron of a triangle, of its edges and of its
// vertices lies inside the triangle's slab box or inside the box of one of its edges grown by the reach rb, so marking
// those four boxes per triangle (corners + normal only) covers every cell the evaluation can touch.
__device__ __forceinline__ void mark_box(const GridParams &g, const float *mn, const float *mx,
                                         unsigned char *__restrict__ brick_flag) {
    // a non-finite corner (the soup is being rejected with SDF_EINVAL anyway) would turn into whole-axis ranges: a thread
    // walking every brick of the grid, per such triangle
    if (!isfinite(mn[0] + mn[1] + mn[2] + mx[0] + mx[1] + mx[2])) return;
    int i0, i1, j0, j1, k0, k1;
    cell_range(mn[0], mx[0], g.ox, g.inv_h, g.nx, i0, i1);
    cell_range(mn[1], mx[1], g.oy, g.inv_h, g.ny, j0, j1);
    cell_range(mn[2], mx[2], g.oz, g.inv_h, g.nz, k0, k1);
    if (!(i0 <= i1 && j0 <= j1 && k0 <= k1)) return;
    for (int bz = k0 >> 3; bz <= (k1 >> 3); bz++)
        for (int by = j0 >> 3; by <= (j1 >> 3); by++)
            for (int bx = i0 >> 3; bx <= (i1 >> 3); bx++) {
                unsigned char *f = brick_flag + ((size_t)bz * g.nby + by) * g.nbx + bx;
                if (!*f) *f = 1;            // mostly already set: a cached read, not a write
            }
}
// A small triangle (or the AABB debug mode): its box grown by the reach holds all four boxes and costs no extra brick.
// Marks it and returns true; false for a larger triangle (nothing marked).
__device__ __forceinline__ bool mark_triangle_small(const GridParams &g, const float *T,
                                                    unsigned char *__restrict__ brick_flag) {
    const float rb = g.rb, eps = g.eps;
    float lo[3], hi[3], mn[3], mx[3];
    float ext_max = 0.0f;
#pragma unroll
    for (int i = 0; i < 3; i++) {
        lo[i] = fminf(T[i], fminf(T[3 + i], T[6 + i])); hi[i] = fmaxf(T[i], fmaxf(T[3 + i], T[6 + i]));
        ext_max = fmaxf(ext_max, hi[i] - lo[i]);
    }
    if (!(g.aabb_mode || ext_max <= 4.0f * g.h)) return false;
#pragma unroll
    for (int i = 0; i < 3; i++) { mn[i] = lo[i] - rb - eps; mx[i] = hi[i] + rb + eps; }
    mark_box(g, mn, mx, brick_flag);
    return true;
}
// box q of a larger triangle: 0 = the slab box, 1..3 = the box of edge q-1 grown by the reach
__device__ __forceinline__ void triangle_part_box(const GridParams &g, const float *T, const float *N, int q,
                                                  float *mn, float *mx) {
    const float rb = g.rb, eps = g.eps;
    if (q == 0) {
#pragma unroll
        for (int i = 0; i < 3; i++) {
            const float lo = fminf(T[i], fminf(T[3 + i], T[6 + i])), hi = fmaxf(T[i], fmaxf(T[3 + i], T[6 + i]));
            const float ext = rb * fabsf(N[i]);
            mn[i] = lo - ext - eps; mx[i] = hi + ext + eps;
        }
    } else {
        const int k = q - 1;
        const float *A = T + 3 * k, *B = T + 3 * (k == 2 ? 0 : k + 1);
#pragma unroll
        for (int i = 0; i < 3; i++) {
            mn[i] = fminf(A[i], B[i]) - rb - eps;
            mx[i] = fmaxf(A[i], B[i]) + rb + eps;
        }
    }
}
// one thread, all boxes (tri_geom_kernel: C4-like meshes of sub-cell triangles, one box each)
__device__ __forceinline__ void mark_triangle_bricks(const GridParams &g, const float *T, const float *N,
                                                     unsigned char *__restrict__ brick_flag) {
    if (mark_triangle_small(g, T, brick_flag)) return;
#pragma unroll
    for (int q = 0; q < 4; q++) {
        float mn[3], mx[3];
        triangle_part_box(g, T, N, q, mn, mx);
        mark_box(g, mn, mx, brick_flag);
    }
}

// Face slab p: sine of its sideways margin = the widest smooth edge (fsm, from the edge pass) or smooth vertex (vsm: one
// byte per vertex, rounded up) it absorbs.  Three byte gathers per face, inside the instruction-bound evaluate kernels.
__device__ __forceinline__ float face_margin_sin(const MeshView &mv, int64_t p) {
    float s = mv.fsm[p];
    u32 code = 0;
#pragma unroll
    for (int k = 0; k < 3; k++) code = max(code, (u32)mv.vsm[mv.cvid[3 * p + k]]);
    return fmaxf(s, (float)code * (1.0f / VSM_SCALE));
}

// A5: bounding volume of polyhedron p in cell indices, clipped to the grid.  Returns false if
// the polyhedron is not emitted (flat edge, one-sided vertex, skipped cone) or misses the grid.
__device__ __forceinline__ bool poly_aabv(const MeshView &mv, const GridParams &g, int64_t p, PolyHdr &h) {
    float mn[3], mx[3];
    bool emit = true;
    const float rb = g.rb, eps = g.eps;
    if (p < mv.F) {
        // face slab: triangle swept by +-rb along its normal
        const float *T = mv.soup + 9 * p, *N = mv.fn + 3 * p;
        emit = !(g.disable & 1);
        h.msin = emit ? face_margin_sin(mv, p) : 0.0f;
        const float dl = rb * h.msin;               // sideways margin for the smooth edges / vertices it absorbs
#pragma unroll
        for (int i = 0; i < 3; i++) {
            float lo = fminf(T[i], fminf(T[3 + i], T[6 + i])), hi = fmaxf(T[i], fmaxf(T[3 + i], T[6 + i]));
            float ext = g.aabb_mode ? rb : rb * fabsf(N[i]) + dl;
            mn[i] = lo - ext - eps; mx[i] = hi + ext + eps;
        }
    } else if (p < (int64_t)mv.F + mv.E) {
        // edge wedge: segment swept by the arc between n1 and n2, radius rb
        const EdgeRec &r = mv.erec[p - mv.F];
        emit = !g.aabb_mode && !(g.disable & 2);          // every record is a wedge that exists
        if (emit && r.cls == 2) {
            // knife edge: the cylinder of radius rb about the segment
#pragma unroll
            for (int i = 0; i < 3; i++) {
                mn[i] = fminf(r.a[i], r.b[i]) - rb - eps;
                mx[i] = fmaxf(r.a[i], r.b[i]) + rb + eps;
            }
        } else if (emit) {
            // the wedge spans the arc n1 -> n2 on the outside of a convex edge and the arc
            // -n1 -> -n2 on the inside of a concave one
            const float sg = r.cls > 0 ? 1.0f : -1.0f;
            f3 a = ld3(r.a), b = ld3(r.b), n1 = sg * ld3(r.n1), n2 = sg * ld3(r.n2);
            f3 u = b - a;
            u = rsqrtf(dot(u, u)) * u;
            f3 w1 = cross(u, ld3(r.n1)), w2 = cross(ld3(r.n2), u);     // same side planes for both classes
            const float A[3] = {a.x, a.y, a.z}, B[3] = {b.x, b.y, b.z}, U[3] = {u.x, u.y, u.z};
            const float N1[3] = {n1.x, n1.y, n1.z}, N2[3] = {n2.x, n2.y, n2.z};
            const float W1[3] = {w1.x, w1.y, w1.z}, W2[3] = {w2.x, w2.y, w2.z};
#pragma unroll
            for (int i = 0; i < 3; i++) {
                float pk = sqrtf(fmaxf(0.0f, 1.0f - U[i] * U[i]));   // axis i projected on the plane normal to u
                float up = fmaxf(0.0f, fmaxf(N1[i], N2[i]));
                float dn = fminf(0.0f, fminf(N1[i], N2[i]));
                if (W1[i] >= -1e-5f && W2[i] >= -1e-5f) up = fmaxf(up, pk);    // +axis direction inside the arc
                if (W1[i] <= 1e-5f && W2[i] <= 1e-5f) dn = fminf(dn, -pk);     // -axis direction inside the arc
                mn[i] = fminf(A[i], B[i]) + rb * dn - eps;
                mx[i] = fmaxf(A[i], B[i]) + rb * up + eps;
            }
        }
    } else {
        // vertex cone about +-pseudonormal intersected with the ball of radius rb
        // (cone AABV intersected with the sphere AABV)
        const u32 q = mv.cone_list[p - mv.F - mv.E];
        const VertexRec &r = mv.vrec[q >> 1];
        int side = (int)(q & 1);
        emit = !g.aabb_mode && !(g.disable & 4);          // every entry is a cone that exists
        if (emit) {
            float sg = side ? -1.0f : 1.0f;
            float c = r.cos_cone, sn = sqrtf(fmaxf(0.0f, 1.0f - c * c));
#pragma unroll
            for (int i = 0; i < 3; i++) {
                float ai = sg * r.axis[i], pk = sqrtf(fmaxf(0.0f, 1.0f - ai * ai));
                float up = (ai >= c) ? 1.0f : fmaxf(0.0f, ai * c + pk * sn + 1e-6f);
                float dn = (-ai >= c) ? -1.0f : fminf(0.0f, ai * c - pk * sn - 1e-6f);
                mn[i] = r.pos[i] + rb * dn - eps;
                mx[i] = r.pos[i] + rb * up + eps;
            }
        }
    }
    h.i0 = h.j0 = h.k0 = 0; h.i1 = h.j1 = h.k1 = -1; h.rows = 0;
    if (p >= mv.F) h.msin = 0.0f;
    if (!emit) return false;
    int i0, i1, j0, j1, k0, k1;
    cell_range(mn[0], mx[0], g.ox, g.inv_h, g.nx, i0, i1);
    cell_range(mn[1], mx[1], g.oy, g.inv_h, g.ny, j0, j1);
    cell_range(mn[2], mx[2], g.oz, g.inv_h, g.nz, k0, k1);
    if (!(i0 <= i1 && j0 <= j1 && k0 <= k1)) return false;
    h.i0 = (short)i0; h.i1 = (short)i1; h.j0 = (short)j0; h.j1 = (short)j1; h.k0 = (short)k0; h.k1 = (short)k1;
    h.rows = (u32)(j1 - j0 + 1) * (u32)(k1 - k0 + 1);
    return true;
}

// Sign carried with the candidate (the polarity of the winning extrusion).  A face
// prism knows the side from n.r, a wedge from its class, a cone from its side; FL_SURE says the
// emit pass may take that sign as is.  Candidates from the eps margin of a prism, from the end
// cap of a wedge, near the dividing plane of a cone / hemisphere or from a knife edge leave it
// clear and the emit pass decides from the pseudonormal of the closest feature.
#define FL_NEG 1u
#define FL_SURE 2u
#define TY_NEG 16        // record type word: bit 4 = interior side, bit 5 = never sure
#define TY_UNSURE 32

// a distance this small against the operands it was differenced from has no reliable sign in fp32
// (relative to the operands of the difference -- and absolutely: a cell coordinate fmaf(i, h, o) carries half an ulp of the
// largest coordinate of the grid whatever the size of r; g.tiny_abs = two such ulps)
__device__ __forceinline__ bool tiny_vs(const GridParams &g, float d, f3 r) {
    return d <= 1e-5f * (fabsf(r.x) + fabsf(r.y) + fabsf(r.z)) || d <= g.tiny_abs;
}

__device__ __forceinline__ void put_min(const GridParams &g, const int *__restrict__ table, u64 *__restrict__ scratch,
                                        int i, int j, int k, float d, int id, u32 fl) {
    int slot = table[((size_t)(k >> 3) * g.nby + (j >> 3)) * g.nbx + (i >> 3)];
    if (slot < 0) return;          // cannot happen: brick_mark_kernel covers every polyhedron
    u64 *cell = scratch + (size_t)slot * BRICK_CELLS + (((k & 7) * 8 + (j & 7)) * 8 + (i & 7));
    // low word: id, then FL_SURE, then FL_NEG -- among equal (d, id) an unsure entry wins
    const u64 val = ((u64)__float_as_uint(d) << 32) | ((u32)id << 2) | fl;
    if (g.scratch_hint) {
        // keep the scratch lines in L2 (evict-last) while the sentinel fill streams past them (evict-first): C4 -0.5 %,
        // C5 -2.2 % of the step (SDF_SCRATCH_HINT=0 switches it off)
        u64 pol;
        asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
        asm volatile("red.global.min.u64.L2::cache_hint [%0], %1, %2;" :: "l"(cell), "l"(val), "l"(pol) : "memory");
    } else {
        atomicMin(cell, val);
    }
}

__device__ __forceinline__ void add_stats(u64 *__restrict__ ctr, u32 tested, u32 accepted, u32 rows) {
    // warp-reduced, spread over CTR_SLOTS lines: same-address atomics serialise in L2
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        tested += __shfl_xor_sync(0xffffffffu, tested, o);
        accepted += __shfl_xor_sync(0xffffffffu, accepted, o);
        rows += __shfl_xor_sync(0xffffffffu, rows, o);
    }
    if ((threadIdx.x & 31) == 0) {
        u64 *s = ctr + CTR_SPREAD + ((blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) & (CTR_SLOTS - 1)) * 8;
        if (tested) atomicAdd(s + SP_TESTED, (u64)tested);
        if (accepted) atomicAdd(s + SP_ACCEPTED, (u64)accepted);
        if (rows) atomicAdd(s + SP_ROWS, (u64)rows);
    }
}

// ---- ABLATION, off by default: the paper's first scheduler, "a single
// thread per extrusion that loops over the cells of its bounding volume" (Table 4).
// The lane that owns the polyhedron walks its bounding volume itself, plane coefficients in
// registers: no record, no search, two FMAs per plane and row, one per plane and cell -- and the
// divergent trip counts of 32 different polyhedra per warp.  SDF_SCHEDULER=serial selects it for
// every polyhedron the block-per-polyhedron kernel does not take; DESIGN.md sec.12 has the numbers.
__device__ __forceinline__ void process_direct(const MeshView &mv, const GridParams &g, int64_t p, const PolyHdr &H,
                                               const int *__restrict__ table, u64 *__restrict__ scratch,
                                               u32 &tested, u32 &accepted) {
    const float h = g.h, eps = g.eps, reach = g.band + g.guard;
    const int i0 = H.i0, j0 = H.j0, k0 = H.k0, ni = H.i1 - H.i0 + 1, nj = H.j1 - H.j0 + 1, nk = H.k1 - H.k0 + 1;
    if (p < mv.F) {
        const float *T = mv.soup + 9 * p, *N = mv.fn + 3 * p;
        const f3 a = ld3(T), e0 = ld3(T + 3) - a, ec = ld3(T + 6) - a, n = ld3(N);
        const f3 e1 = ec - e0;
        const f3 m0 = cross(n, e0), m1 = cross(n, e1), m2 = cross(ec, n);          // inward, |m_i| = |edge_i|
        const float em = eps + g.rb * H.msin;
        const float t0 = em * sqrtf(dot(e0, e0)), t1 = em * sqrtf(dot(e1, e1)), t2 = em * sqrtf(dot(ec, ec));
        const int id = mv.perm[p];
        const f3 r0 = mk<float>(fmaf((float)i0, h, g.ox) - a.x, fmaf((float)j0, h, g.oy) - a.y, fmaf((float)k0, h, g.oz) - a.z);
        const float c0 = dot(m0, r0), c1 = dot(m1, r0) - dot(m1, e0), c2 = dot(m2, r0) - dot(m2, ec), cn = dot(n, r0);
        for (int dk = 0; dk < nk; dk++) {
            const float fk = (float)dk * h;
            const float rz = __fsub_rn(fmaf((float)(k0 + dk), h, g.oz), a.z);
            for (int dj = 0; dj < nj; dj++) {
                const float fj = (float)dj * h;
                const float ry = __fsub_rn(fmaf((float)(j0 + dj), h, g.oy), a.y);
                const float b0 = fmaf(m0.z, fk, fmaf(m0.y, fj, c0)), b1 = fmaf(m1.z, fk, fmaf(m1.y, fj, c1));
                const float b2 = fmaf(m2.z, fk, fmaf(m2.y, fj, c2)), bn = fmaf(n.z, fk, fmaf(n.y, fj, cn));
                for (int di = 0; di < ni; di++) {
                    const float fi = (float)di * h;
                    const float s0 = fmaf(m0.x, fi, b0), s1 = fmaf(m1.x, fi, b1), s2 = fmaf(m2.x, fi, b2);
                    const float dn = fmaf(n.x, fi, bn);
                    if (s0 < -t0 || s1 < -t1 || s2 < -t2 || fabsf(dn) >= reach + eps) continue;
                    const int i = i0 + di;
                    const f3 r = mk<float>(__fsub_rn(fmaf((float)i, h, g.ox), a.x), ry, rz);
                    float d;
                    u32 fl = 0;
                    if (s0 >= 0.0f && s1 >= 0.0f && s2 >= 0.0f) {
                        const float dnc = dot_rn(n, r);
                        d = fabsf(dnc);
                        fl = (tiny_vs(g, d, r) ? 0u : FL_SURE) | (dnc < 0.0f ? FL_NEG : 0u);
                    } else {
                        int rg; f3 qq;                // eps margin: exact clamped distance
                        d = tri_closest<float>(r, e0, ec, n, rg, qq);
                    }
                    if (d < reach) { accepted++; put_min(g, table, scratch, i, j0 + dj, k0 + dk, d, id, fl); }
                }
            }
        }
    } else if (p < (int64_t)mv.F + mv.E) {
        const EdgeRec &er = mv.erec[p - mv.F];
        const f3 a = ld3(er.a), ab = ld3(er.b) - a, n1 = ld3(er.n1), n2 = ld3(er.n2);
        const float L = sqrtf(dot(ab, ab));
        const f3 u = (1.0f / L) * ab;
        f3 w1 = cross(u, n1), w2 = cross(n2, u);
        if (er.cls == 2) w1 = w2 = mk<float>(0.0f, 0.0f, 0.0f);       // knife edge: no side planes
        f3 nbis = n1 + n2;
        nbis = rsqrtf(fmaxf(dot(nbis, nbis), 1e-30f)) * nbis;
        const int id = er.tri;
        const u32 fl_rec = (er.cls < 0 ? FL_NEG : 0u) | ((dot(n1, n2) < -0.99f || er.cls == 2) ? 0u : FL_SURE);
        const f3 r0 = mk<float>(fmaf((float)i0, h, g.ox) - a.x, fmaf((float)j0, h, g.oy) - a.y, fmaf((float)k0, h, g.oz) - a.z);
        const float ct = dot(u, r0), c1 = dot(w1, r0), c2 = dot(w2, r0);
        for (int dk = 0; dk < nk; dk++) {
            const float fk = (float)dk * h;
            const float rz = __fsub_rn(fmaf((float)(k0 + dk), h, g.oz), a.z);
            for (int dj = 0; dj < nj; dj++) {
                const float fj = (float)dj * h;
                const float ry = __fsub_rn(fmaf((float)(j0 + dj), h, g.oy), a.y);
                const float bt = fmaf(u.z, fk, fmaf(u.y, fj, ct)), b1 = fmaf(w1.z, fk, fmaf(w1.y, fj, c1));
                const float b2 = fmaf(w2.z, fk, fmaf(w2.y, fj, c2));
                for (int di = 0; di < ni; di++) {
                    const float fi = (float)di * h;
                    const float t = fmaf(u.x, fi, bt);
                    if (t < -eps || t > L + eps || fmaf(w1.x, fi, b1) < -eps || fmaf(w2.x, fi, b2) < -eps) continue;
                    const int i = i0 + di;
                    const f3 r = mk<float>(__fsub_rn(fmaf((float)i, h, g.ox), a.x), ry, rz);
                    const float tu = dot_rn(u, r), tc = fminf(fmaxf(tu, 0.0f), L);
                    const f3 q = mk<float>(__fmaf_rn(-tc, u.x, r.x), __fmaf_rn(-tc, u.y, r.y), __fmaf_rn(-tc, u.z, r.z));
                    const float d = __fsqrt_rn(dot_rn(q, q));
                    const float sb = (fl_rec & FL_NEG) ? -dot(nbis, q) : dot(nbis, q);
                    const u32 fl = (tu > 0.0f && tu < L && sb > 1e-2f * d && !tiny_vs(g, d, r)) ? fl_rec : (fl_rec & FL_NEG);
                    if (d < reach) { accepted++; put_min(g, table, scratch, i, j0 + dj, k0 + dk, d, id, fl); }
                }
            }
        }
    } else {
        const u32 q = mv.cone_list[p - mv.F - mv.E];
        const VertexRec &vr = mv.vrec[q >> 1];
        const float sg = (q & 1) ? -1.0f : 1.0f;
        const f3 v = ld3(vr.pos), A = sg * ld3(vr.axis);
        const float c = vr.cos_cone;
        const int id = mv.vmint[q >> 1];
        const u32 fl_rec = ((q & 1) ? FL_NEG : 0u) | (c <= -1.0f ? 0u : FL_SURE);
        for (int dk = 0; dk < nk; dk++) {
            const float rz = __fsub_rn(fmaf((float)(k0 + dk), h, g.oz), v.z);
            for (int dj = 0; dj < nj; dj++) {
                const float ry = __fsub_rn(fmaf((float)(j0 + dj), h, g.oy), v.y);
                if (ry * ry + rz * rz >= reach * reach) continue;
                for (int di = 0; di < ni; di++) {
                    const int i = i0 + di;
                    const f3 r = mk<float>(__fsub_rn(fmaf((float)i, h, g.ox), v.x), ry, rz);
                    const float d = __fsqrt_rn(dot_rn(r, r)), ar = dot(A, r);
                    if (d >= reach || ar < c * d - eps) continue;
                    accepted++;
                    put_min(g, table, scratch, i, j0 + dj, k0 + dk, d, id, (ar > 1e-2f * d && !tiny_vs(g, d, r)) ? fl_rec : (fl_rec & FL_NEG));
                }
            }
        }
    }
    tested += (u32)(ni * nj * nk);
}

// cdp.cu (ablation): A5-A7 with the paper's dynamic-parallelism scheduler instead of the two
// evaluate kernels; same scratch, same candidates
int run_cdp_evaluate(sdf_mesh *m, const MeshView &mv, const GridParams &g, cudaStream_t st);
