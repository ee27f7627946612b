// compute.cu -- sdf_compute: clip the characteristic polyhedra to band + grid (A5), count
// their grid rows and prefix-sum them into flat work items (A6), evaluate exact feature
// distances with a packed 64-bit atomicMin into band-sparse bricks (A7), then sign and emit
// the dense grids (A8).
//
//   A5  PAPER.md:344-364 (sec.8: prisms, wedges, cones/hemispheres and their AABVs)
//   A6  PAPER.md:242-252 (sec.5: half-plane scan conversion) -- replaces the schedulers of
//       PAPER.md:366-380 (thread per extrusion / dynamic parallelism) by count -> scan -> items
//   A7  PAPER.md:63-77, 374, 386-392 (min-magnitude combine, eps-tolerant inclusion tests,
//       feature distances)
//   A8  PAPER.md:217 (sign from the angle-weighted pseudonormal of the closest feature),
//       PAPER.md:66, 392 (infinity outside the band)
#include "primitives.cuh"
#include <math.h>

#include "evaluate.cuh"

// A6a (evaluate.cuh): four threads per triangle.  The first decides whether the triangle is small (one box of a few
// bricks: it marks them, the other three leave after one shuffle); the four boxes of a larger one go to one thread each
// (one thread walking all four in turn: 56 us for the 20480 triangles of C2, 0.2 ms at C5; the whole warp walking one
// triangle's boxes after another was tried too and is slower still: C3 0.41 -> 0.47 ms).
// SPLIT = false: a thread per triangle does it all (meshes of millions of sub-cell triangles, where three of the four
// threads would only add waves).
template <bool SPLIT>
__global__ void __launch_bounds__(256) brick_mark_kernel(MeshView mv, GridParams g,
                                                         unsigned char *__restrict__ brick_flag) {
    const int64_t gid = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (!SPLIT) {
        if (gid < mv.F) mark_triangle_bricks(g, mv.soup + 9 * gid, mv.fn + 3 * gid, brick_flag);
        return;
    }
    const int64_t t = gid >> 2;
    const int q = (int)(gid & 3), lane = threadIdx.x & 31;
    const bool valid = t < mv.F;
    float T[9], N[3];
    int small = 1;
    if (valid && q == 0) {
#pragma unroll
        for (int i = 0; i < 9; i++) T[i] = mv.soup[9 * t + i];
        small = mark_triangle_small(g, T, brick_flag) ? 1 : 0;
    }
    small = __shfl_sync(0xffffffffu, small, lane & ~3);
    if (small || !valid) return;
    if (q) {
#pragma unroll
        for (int i = 0; i < 9; i++) T[i] = mv.soup[9 * t + i];
    }
#pragma unroll
    for (int i = 0; i < 3; i++) N[i] = mv.fn[3 * t + i];
    float mn[3], mx[3];
    triangle_part_box(g, T, N, q, mn, mx);
    mark_box(g, mn, mx, brick_flag);
}

struct BrickIn {
    const unsigned char *flag;
    __device__ u64 operator()(int64_t i) const { return flag[i]; }
};
struct BrickOut {
    int *table, *list;        // brick -> scratch slot (-1 = inactive), slot -> brick
    __device__ void operator()(int64_t i, u64 ex, u64 v) const {
        table[i] = v ? (int)ex : -1;
        if (v) list[ex] = (int)i;
    }
};

// ---------------------------------------------------------------------------------------
// A6 + A7: scan conversion and evaluation.
//
// A polyhedron is turned into a 29-word record in shared memory: its planes in the form the row
// walk needs (a convex body meets a grid row in one interval, and along the row every half-space
// test s = base + di * g is linear in the cell index), the triangle id, the sign
// flags and the AABV.  Work is flattened WITHIN A WARP: lane l owns polyhedron 32*warp + l, the
// row counts are prefix-summed across the lanes, and the warp then walks the flattened
// (polyhedron, row) list 32 rows at a time -- the load balancing of PAPER.md:376-380 (dynamic
// parallelism) without child launches, without a global work-item list and without a device-wide
// scan.  Polyhedra with many or long rows are listed by evaluate_small_kernel and taken by
// evaluate_big_kernel, one block per polyhedron: a thread per row when there are many rows, a
// warp per row with the lanes along x when there are few long ones.
// ---------------------------------------------------------------------------------------
// ---- small polyhedra: compact record + incremental scan conversion of a grid row.
// Along a grid row every half-space test of PAPER.md:246-252 is linear in the cell index,
// s(di) = base + di * g, so a row costs one set-up (the j,k terms) and one FMA + compare per
// plane and cell; rows longer than g.row_clip cells (2; SDF_ROW_CLIP) are first clipped analytically (a convex
// body meets a line in one interval).  Cells that pass get the distance from the canonical
// expressions (cell position by one fmaf, differences first, dot_rn), so a distance does not
// depend on which path evaluated it.
#define RR_ID 20
#define RR_TYPE 21
#define RR_I0 22
#define RR_J0 23
#define RR_K0 24
#define RR_NI 25
#define RR_NJ 26
#define RR_INV_NJ 27     // float 1 / nj
#define RR_TIDX 28       // faces: internal triangle index (the eps-margin path re-reads the corners)
#define RR_WORDS 29      // odd stride: records of different owners fall in different banks

__device__ __forceinline__ void build_row_record(const MeshView &mv, const GridParams &g, int64_t p, const PolyHdr &H,
                                                 float *rec) {
    const float eps = g.eps;
    int *ri = (int *)rec;
    if (p < mv.F) {
        // face slab: three inward side planes through the edges + the slab
        const float *T = mv.soup + 9 * p, *N = mv.fn + 3 * p;
        const f3 a = ld3(T), e0 = ld3(T + 3) - a, ec = ld3(T + 6) - a, n = ld3(N);
        const f3 e1 = ec - e0;
        const f3 m0 = cross(n, e0), m1 = cross(n, e1), m2 = cross(ec, n);          // inward, |m_i| = |edge_i|
        rec[0] = a.x; rec[1] = a.y; rec[2] = a.z; rec[3] = n.x; rec[4] = n.y; rec[5] = n.z;
        rec[6] = m0.x; rec[7] = m0.y; rec[8] = m0.z; rec[9] = m1.x; rec[10] = m1.y; rec[11] = m1.z;
        rec[12] = m2.x; rec[13] = m2.y; rec[14] = m2.z;
        rec[15] = dot(m1, e0); rec[16] = dot(m2, ec);
        const float em = eps + g.rb * H.msin;          // eps + the margin for absorbed smooth features
        rec[17] = em * sqrtf(dot(e0, e0)); rec[18] = em * sqrtf(dot(e1, e1)); rec[19] = em * sqrtf(dot(ec, ec));
        ri[RR_ID] = mv.perm[p]; ri[RR_TYPE] = 0; ri[RR_TIDX] = (int)p;
    } else if (p < (int64_t)mv.F + mv.E) {
        // edge wedge: beyond both faces' side planes, between the end caps
        const EdgeRec &r = mv.erec[p - mv.F];
        const f3 a = ld3(r.a), ab = ld3(r.b) - a, n1 = ld3(r.n1), n2 = ld3(r.n2);
        const float L = sqrtf(dot(ab, ab));
        const f3 u = (1.0f / L) * ab;
        f3 w1 = cross(u, n1), w2 = cross(n2, u);
        if (r.cls == 2) w1 = w2 = mk<float>(0.0f, 0.0f, 0.0f);        // knife edge: no side planes
        rec[0] = a.x; rec[1] = a.y; rec[2] = a.z; rec[3] = u.x; rec[4] = u.y; rec[5] = u.z; rec[6] = L;
        rec[7] = w1.x; rec[8] = w1.y; rec[9] = w1.z; rec[10] = w2.x; rec[11] = w2.y; rec[12] = w2.z;
        ri[RR_ID] = r.tri;
        ri[RR_TYPE] = 1 | (r.cls < 0 ? TY_NEG : 0) | ((dot(n1, n2) < -0.99f || r.cls == 2) ? TY_UNSURE : 0);
        {
            const f3 nb = n1 + n2;
            const float il = rsqrtf(fmaxf(dot(nb, nb), 1e-30f));
            rec[13] = il * nb.x; rec[14] = il * nb.y; rec[15] = il * nb.z;
        }
    } else {
        // vertex cone / hemisphere (eq.10, 362-364) inside the ball of radius reach
        const u32 q = mv.cone_list[p - mv.F - mv.E];
        const VertexRec &r = mv.vrec[q >> 1];
        const float sg = (q & 1) ? -1.0f : 1.0f;
        rec[0] = r.pos[0]; rec[1] = r.pos[1]; rec[2] = r.pos[2];
        rec[3] = sg * r.axis[0]; rec[4] = sg * r.axis[1]; rec[5] = sg * r.axis[2]; rec[6] = r.cos_cone;
        ri[RR_ID] = mv.vmint[q >> 1];
        ri[RR_TYPE] = 2 | ((q & 1) ? TY_NEG : 0) | (r.cos_cone <= -1.0f ? TY_UNSURE : 0);
    }
    const int nj = H.j1 - H.j0 + 1;
    ri[RR_I0] = H.i0; ri[RR_J0] = H.j0; ri[RR_K0] = H.k0; ri[RR_NI] = H.i1 - H.i0 + 1; ri[RR_NJ] = nj;
    rec[RR_INV_NJ] = 1.0f / (float)nj;
}

// clip the cell-index interval [lo, hi] of a row against base + di * g >= -tol
__device__ __forceinline__ void clip_lin(float base, float gx, float tol, float &lo, float &hi) {
    const float num = -tol - base;
    if (gx > 0.0f) lo = fmaxf(lo, __fdividef(num, gx) - 1e-2f);
    else if (gx < 0.0f) hi = fminf(hi, __fdividef(num, gx) + 1e-2f);
    else if (num > 0.0f) hi = -1.0f;
}

// STRIDE 1: a lane owns the row (small polyhedra); STRIDE 32: a warp does, lane0 = its lane (big ones)
template <int STRIDE, bool EXACT_DIV>
__device__ __forceinline__ void process_row_inc(const MeshView &mv, const GridParams &g, const float *rec, int row,
                                                int lane0, const int *__restrict__ table, u64 *__restrict__ scratch,
                                                u32 &tested, u32 &accepted) {
    const int *ri = (const int *)rec;
    const int nj = ri[RR_NJ], ni = ri[RR_NI], i0 = ri[RR_I0], tyw = ri[RR_TYPE], type = tyw & 15, id = ri[RR_ID];
    const u32 fl_rec = ((tyw & TY_NEG) ? FL_NEG : 0u) | ((tyw & TY_UNSURE) ? 0u : FL_SURE);
    // rows of a small polyhedron (<= 256) divide exactly through the fp32 reciprocal
    const int dk = EXACT_DIV ? row / nj : (int)(((float)row + 0.5f) * rec[RR_INV_NJ]);
    const int j = ri[RR_J0] + row - dk * nj, k = ri[RR_K0] + dk;
    const float h = g.h, eps = g.eps, reach = g.band + g.guard;      // accept d < reach; the emit pass decides exactly
    const float ry = __fsub_rn(fmaf((float)j, h, g.oy), rec[1]), rz = __fsub_rn(fmaf((float)k, h, g.oz), rec[2]);
    const float rx0 = fmaf((float)i0, h, g.ox) - rec[0];
    int da = 0, db = ni - 1;
    if (type == 0) {
        const f3 n = ld3(rec + 3), m0 = ld3(rec + 6), m1 = ld3(rec + 9), m2 = ld3(rec + 12);
        const float t0 = rec[17], t1 = rec[18], t2 = rec[19];
        const float b0 = fmaf(m0.x, rx0, fmaf(m0.y, ry, m0.z * rz)), g0 = m0.x * h;
        const float b1 = fmaf(m1.x, rx0, fmaf(m1.y, ry, m1.z * rz)) - rec[15], g1 = m1.x * h;
        const float b2 = fmaf(m2.x, rx0, fmaf(m2.y, ry, m2.z * rz)) - rec[16], g2 = m2.x * h;
        const float bn = fmaf(n.x, rx0, fmaf(n.y, ry, n.z * rz)), gn = n.x * h;
        if (ni > g.row_clip && !g.aabb_mode) {
            float lo = 0.0f, hi = (float)db;
            clip_lin(b0, g0, t0, lo, hi); clip_lin(b1, g1, t1, lo, hi); clip_lin(b2, g2, t2, lo, hi);
            clip_lin(bn, gn, reach, lo, hi); clip_lin(-bn, -gn, reach, lo, hi);
            if (!(lo <= hi)) return;
            da = (int)ceilf(lo); db = (int)floorf(hi);
        }
        for (int di = da + lane0; di <= db; di += STRIDE) {
            const float fd = (float)di;
            const float s0 = fmaf(fd, g0, b0), s1 = fmaf(fd, g1, b1), s2 = fmaf(fd, g2, b2), dn = fmaf(fd, gn, bn);
            tested++;
            // debug mode "AABB candidates": every cell of the band-expanded box gets the clamped distance
            if (!g.aabb_mode && (s0 < -t0 || s1 < -t1 || s2 < -t2 || fabsf(dn) >= reach + eps)) continue;
            const int i = i0 + di;
            const f3 r = mk<float>(__fsub_rn(fmaf((float)i, h, g.ox), rec[0]), ry, rz);
            float d;
            u32 fl = 0;
            if (s0 >= 0.0f && s1 >= 0.0f && s2 >= 0.0f && !g.aabb_mode) {
                const float dnc = dot_rn(n, r);
                d = fabsf(dnc);
                fl = (tiny_vs(g, d, r) ? 0u : FL_SURE) | (dnc < 0.0f ? FL_NEG : 0u);
            } else {
                // eps margin: exact clamped distance from the triangle itself
                const float *T = mv.soup + 9 * (size_t)ri[RR_TIDX];
                const f3 a = ld3(T);
                int rg; f3 qq;
                d = tri_closest<float>(r, ld3(T + 3) - a, ld3(T + 6) - a, n, rg, qq);
            }
            if (d < reach) { accepted++; put_min(g, table, scratch, i, j, k, d, id, fl); }
        }
    } else if (type == 1) {
        const f3 u = ld3(rec + 3), w1 = ld3(rec + 7), w2 = ld3(rec + 10), nbis = ld3(rec + 13);
        const float L = rec[6];
        const float bt = fmaf(u.x, rx0, fmaf(u.y, ry, u.z * rz)), gt = u.x * h;
        const float b1 = fmaf(w1.x, rx0, fmaf(w1.y, ry, w1.z * rz)), g1 = w1.x * h;
        const float b2 = fmaf(w2.x, rx0, fmaf(w2.y, ry, w2.z * rz)), g2 = w2.x * h;
        if (ni > g.row_clip) {
            float lo = 0.0f, hi = (float)db;
            clip_lin(bt, gt, eps, lo, hi); clip_lin(L - bt, -gt, eps, lo, hi);
            clip_lin(b1, g1, eps, lo, hi); clip_lin(b2, g2, eps, lo, hi);
            if (!(lo <= hi)) return;
            da = (int)ceilf(lo); db = (int)floorf(hi);
        }
        for (int di = da + lane0; di <= db; di += STRIDE) {
            const float fd = (float)di;
            const float t = fmaf(fd, gt, bt);
            tested++;
            if (t < -eps || t > L + eps || fmaf(fd, g1, b1) < -eps || fmaf(fd, g2, b2) < -eps) continue;
            const int i = i0 + di;
            const f3 r = mk<float>(__fsub_rn(fmaf((float)i, h, g.ox), rec[0]), ry, rz);
            const float tu = dot_rn(u, r), tc = fminf(fmaxf(tu, 0.0f), L);
            const f3 q = mk<float>(__fmaf_rn(-tc, u.x, r.x), __fmaf_rn(-tc, u.y, r.y), __fmaf_rn(-tc, u.z, r.z));
            const float d = __fsqrt_rn(dot_rn(q, q));
            // the end caps belong to the end vertices, and the eps slack of a nearly flat wedge
            // reaches through the surface: the class gives the sign only where the bisector agrees
            const float sb = (fl_rec & FL_NEG) ? -dot(nbis, q) : dot(nbis, q);
            const u32 fl = (tu > 0.0f && tu < L && sb > 1e-2f * d && !tiny_vs(g, d, r)) ? fl_rec : (fl_rec & FL_NEG);
            if (d < reach) { accepted++; put_min(g, table, scratch, i, j, k, d, id, fl); }
        }
    } else {
        const f3 A = ld3(rec + 3);
        const float c = rec[6];
        // ball of radius reach about the vertex: |rx| <= xr on this row
        const float rem = reach * reach - ry * ry - rz * rz;
        if (rem < 0.0f) return;
        const float xr = sqrtf(rem);
        float lo = fmaxf(0.0f, (-xr - rx0) * g.inv_h - 1e-2f), hi = fminf((float)db, (xr - rx0) * g.inv_h + 1e-2f);
        // a cone of half angle <= 90 degrees lies in the half space A.r >= 0
        const float ba = fmaf(A.x, rx0, fmaf(A.y, ry, A.z * rz)), ga = A.x * h;
        if (c >= 0.0f) clip_lin(ba, ga, 2.0f * eps, lo, hi);
        if (!(lo <= hi)) return;
        da = (int)ceilf(lo); db = (int)floorf(hi);
        for (int di = da + lane0; di <= db; di += STRIDE) {
            const int i = i0 + di;
            const f3 r = mk<float>(__fsub_rn(fmaf((float)i, h, g.ox), rec[0]), ry, rz);
            tested++;
            const float d = __fsqrt_rn(dot_rn(r, r)), ar = dot(A, r);
            if (d >= reach || ar < c * d - eps) continue;
            accepted++;
            // near the plane through the vertex normal to the axis the side is not decided here
            put_min(g, table, scratch, i, j, k, d, id, (ar > 1e-2f * d && !tiny_vs(g, d, r)) ? fl_rec : (fl_rec & FL_NEG));
        }
    }
}

// The order in which the warps of evaluate_small_kernel take the polyhedra.  The index space is [faces | wedges | cones],
// each class roughly along the Morton order of the triangles; taken front to back the grid is swept three times and a
// scratch sector has left L2 (the sentinel fill streams through it meanwhile) before the next class comes by.  So the
// warps are dealt out in `chunks` rounds: round k takes the k-th part of the faces, of the wedges and of the cones --
// one sweep over space, the three classes of a region close together in time.
struct EvalOrder {
    int64_t chunks;         // 0: plain order
    int64_t wf, we, wc;     // warps per round for faces / wedges / cones
    __device__ __forceinline__ int64_t poly_of(int64_t W, int ppw, int lane, const MeshView &mv) const {
        if (lane >= ppw) return -1;
        if (!chunks) {
            const int64_t p = W * ppw + lane;
            return p < mv.P ? p : -1;
        }
        const int64_t per = wf + we + wc, k = W / per, r = W - k * per;
        int64_t lo, hi, wi;
        if (r < wf) { wi = k * wf + r; lo = 0; hi = mv.F; }
        else if (r < wf + we) { wi = k * we + (r - wf); lo = mv.F; hi = (int64_t)mv.F + mv.E; }
        else { wi = k * wc + (r - wf - we); lo = (int64_t)mv.F + mv.E; hi = mv.P; }
        const int64_t p = lo + wi * ppw + lane;
        return p < hi ? p : -1;
    }
};

#define ES_WARPS 4
#ifndef ES_MINB
#define ES_MINB 9
#endif
template <bool SERIAL>
__global__ void __launch_bounds__(32 * ES_WARPS, SERIAL ? 1 : ES_MINB) evaluate_small_kernel(MeshView mv, GridParams g,
                                                                       u32 *__restrict__ big_list,
                                                                       const int *__restrict__ table,
                                                                       u64 *__restrict__ scratch, u64 *__restrict__ ctr,
                                                                       int ppw, EvalOrder eo) {
    // ppw = polyhedra per warp: 32, or fewer when the mesh has few polyhedra (more warps for the
    // same rows: a mesh of 1e5 medium polyhedra otherwise leaves each scheduler 5 long-running warps)
    __shared__ float s_rec[ES_WARPS][32][RR_WORDS];
    __shared__ int s_ex[ES_WARPS][33];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t p = eo.poly_of((int64_t)blockIdx.x * ES_WARPS + w, ppw, lane, mv);
    int rows = 0;
    bool live = false, direct = false;
    PolyHdr Hd;
    if (p >= 0) {
        PolyHdr H;
        live = poly_aabv(mv, g, p, H);
        if (live) {
            // big polyhedra (many rows or long rows) go to the block-per-polyhedron kernel
            if (H.rows > (u32)g.big_rows || H.i1 - H.i0 >= g.big_ni || g.aabb_mode) {
                big_list[atomicAdd(&ctr[CTR_BIG], 1ull)] = (u32)p;
            } else if (SERIAL) {
                direct = true;
                Hd = H;
            } else {
                rows = (int)H.rows;
                build_row_record(mv, g, p, H, s_rec[w][lane]);
            }
        }
    }
    u32 tested = 0, accepted = 0, rows_direct = 0;
    if (SERIAL && direct) { process_direct(mv, g, p, Hd, table, scratch, tested, accepted); rows_direct = Hd.rows; }
    const unsigned nlive = __popc(__ballot_sync(0xffffffffu, live));
    if (lane == 0 && nlive)
        atomicAdd(&ctr[CTR_SPREAD + ((blockIdx.x * ES_WARPS + w) & (CTR_SLOTS - 1)) * 8 + SP_POLY], (u64)nlive);
    int inc = rows;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
    }
    const int total = __shfl_sync(0xffffffffu, inc, 31);
    s_ex[w][lane] = inc - rows;
    if (lane == 31) s_ex[w][32] = total;
    __syncwarp();
    for (int base = 0; base < total; base += 32) {
        const int r = base + lane;
        if (r < total) {
            int o = 0;                       // largest o with s_ex[o] <= r: the owner of row r
#pragma unroll
            for (int st = 16; st; st >>= 1)
                if (s_ex[w][o + st] <= r) o += st;
            process_row_inc<1, false>(mv, g, s_rec[w][o], r - s_ex[w][o], 0, table, scratch, tested, accepted);
        }
    }
    add_stats(ctr, tested, accepted, (u32)rows + rows_direct);
}

// One block per big polyhedron (dynamic fetch): warps stride over its rows, lanes over x.
#define EBIG_BT 256
#define EBIG_THREAD_ROWS 128      // a big polyhedron with at least this many rows is walked a thread per row
#define EBIG_SPLIT 8             // row slices per big polyhedron when the mesh has few polyhedra
__global__ void __launch_bounds__(EBIG_BT) evaluate_big_kernel(MeshView mv, GridParams g,
                                                               const u32 *__restrict__ big_list,
                                                               const int *__restrict__ table,
                                                               u64 *__restrict__ scratch, u64 *__restrict__ ctr) {
    __shared__ float s_rec[RR_WORDS];
    __shared__ u64 s_e;
    __shared__ u32 s_rows;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const u64 nbig = ctr[CTR_BIG];
    u32 tested = 0, accepted = 0, rows_done = 0;
    while (true) {
        __syncthreads();
        // blockIdx.y = slice: every polyhedron is taken once per slice, and slice y does the
        // row groups y, y + EBIG_SPLIT, ... (a few huge polyhedra, C1, still fill the GPU)
        if (threadIdx.x == 0) s_e = atomicAdd(&ctr[CTR_BIGCUR + blockIdx.y], 1ull);
        __syncthreads();
        const u64 e = s_e;
        if (e >= nbig) break;
        if (threadIdx.x == 0) {
            const int64_t p = (int64_t)big_list[e];
            PolyHdr H;
            poly_aabv(mv, g, p, H);
            build_row_record(mv, g, p, H, s_rec);
            s_rows = H.rows;
        }
        __syncthreads();
        const u32 rows = s_rows;
        if (rows >= EBIG_THREAD_ROWS) {
            // many rows: a thread per row (the row set-up is paid once per row, not once per lane)
            for (u32 r = blockIdx.y * EBIG_BT + threadIdx.x; r < rows; r += gridDim.y * EBIG_BT)
                process_row_inc<1, true>(mv, g, s_rec, (int)r, 0, table, scratch, tested, accepted);
        } else {
            // few, long rows: a warp per row, lanes along x
            for (u32 r = blockIdx.y * (EBIG_BT / 32) + (u32)w; r < rows; r += gridDim.y * (EBIG_BT / 32))
                process_row_inc<32, true>(mv, g, s_rec, (int)r, lane, table, scratch, tested, accepted);
        }
        if (threadIdx.x == 0 && blockIdx.y == 0) rows_done += rows;
    }
    add_stats(ctr, tested, accepted, rows_done);
}

// ---------------------------------------------------------------------------------------
// A8: sign + emit.  Two kernels: (1) fill_tma_kernel (fill_kernel for unaligned outputs) streams the sentinels (+inf, -1;
// PAPER.md:66) over both dense grids at HBM write speed -- it depends on nothing, so it
// runs on a side stream underneath A5-A7; (2) emit_bricks_kernel then overwrites the cells
// of the active bricks: sign from the pseudonormal of the closest feature.
// ---------------------------------------------------------------------------------------
#define FILL_BT 512
#define FILL_UNROLL 4

__global__ void __launch_bounds__(FILL_BT) fill_kernel(float *__restrict__ dist, int *__restrict__ tri, int64_t n,
                                                       int vec) {
    const int64_t tid = (int64_t)blockIdx.x * FILL_BT + threadIdx.x, nth = (int64_t)gridDim.x * FILL_BT;
    if (vec) {
        const int64_t n4 = n >> 2;
        const float4 dv = make_float4(INFINITY, INFINITY, INFINITY, INFINITY);
        const int4 tv = make_int4(-1, -1, -1, -1);
        float4 *d4 = (float4 *)dist;
        int4 *t4 = (int4 *)tri;
        // each block walks contiguous chunks of FILL_UNROLL * FILL_BT vectors (32 KiB per array)
        const int64_t chunk = (int64_t)FILL_BT * FILL_UNROLL;
        for (int64_t base = (int64_t)blockIdx.x * chunk; base < n4; base += (int64_t)gridDim.x * chunk) {
#pragma unroll
            for (int u = 0; u < FILL_UNROLL; u++) {
                int64_t i = base + (int64_t)u * FILL_BT + threadIdx.x;
                if (i < n4) { __stcs(d4 + i, dv); __stcs(t4 + i, tv); }
            }
        }
        for (int64_t i = (n4 << 2) + tid; i < n; i += nth) { dist[i] = INFINITY; tri[i] = -1; }
    } else {
        for (int64_t i = tid; i < n; i += nth) { dist[i] = INFINITY; tri[i] = -1; }
    }
}

// TMA variant (the default): one CTA per SM keeps two sentinel tiles (8 KiB each by default) in shared memory and
// one lane streams them to HBM with bulk asynchronous copies (cp.async.bulk, SASS UBLKCP), L2 evict-first.  It
// needs 4 warps and 16-32 KiB of shared memory per SM, so the kernels of A5-A7 keep (almost) the whole SM while
// 8 B/cell stream out underneath them.
#define FILL_TMA_BT 128
// bytes per bulk copy: runtime, bits 16.. of the `issuers` argument hold log2 (SDF_FILL_CHUNK_LOG2, default 13); issuing
// lanes = bits 0..7 (SDF_FILL_ISSUERS, default 1); pairs in flight per lane = DEPTH + 1 (SDF_FILL_DEPTH, default 2).
// What matters beside another kernel is how many bulk stores are queued in L2 at a time: with one lane the fill both
// runs faster alone (1.18 against 1.22 ms at C4) and holds the evaluate kernels up less (profiles/r2_ablations.md).
// fill_state: [0] = next batch (dynamic fetch), [1 + smid] = SM already has a fill CTA.  More
// CTAs than SMs are launched and the first to arrive on an SM claims it; the others exit at
// once.  (With one CTA per SM by count only, a busy GPU stacked several fill CTAs on the few
// SMs that had room and the fill ran at a fraction of the HBM rate.)
#define FILL_TMA_MAX 16384
#define FILL_BATCH_BYTES 1048576                // bytes per fetch: 1 MiB contiguous per array
#define FILL_STATE_WORDS 1024
template <int DEPTH>
__global__ void __launch_bounds__(FILL_TMA_BT) fill_tma_kernel(float *__restrict__ dist, int *__restrict__ tri,
                                                               int64_t n, int issuers, int batch, u32 *__restrict__ state,
                                                               u32 pat_d, u32 pat_t) {
    __shared__ __align__(128) u32 s_d[FILL_TMA_MAX / 4];
    __shared__ __align__(128) u32 s_t[FILL_TMA_MAX / 4];
    const int chunk = 1 << ((issuers >> 16) & 31);
    __shared__ int s_go;
    const int64_t per = chunk / 4;
    const int64_t nchunks = n / per;
    if (threadIdx.x == 0) {
        u32 smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        s_go = (smid < FILL_STATE_WORDS - 1) ? (atomicCAS(&state[1 + smid], 0u, 1u) == 0u) : 1;
        // throttle (ablation): only sm_share of every 8 SMs stream
        if ((int)(smid & 7u) >= ((issuers >> 8) & 255)) s_go = 0;
    }
    issuers &= 255;
    // ragged tail (< one chunk) with plain stores
    if (blockIdx.x == 0)
        for (int64_t i = nchunks * per + threadIdx.x; i < n; i += FILL_TMA_BT) {
            dist[i] = __uint_as_float(pat_d); tri[i] = (int)pat_t;
        }
    __syncthreads();
    if (!s_go) return;
    for (int i = threadIdx.x; i < chunk / 4; i += FILL_TMA_BT) { s_d[i] = pat_d; s_t[i] = pat_t; }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic-proxy writes -> async proxy reads
    __syncthreads();
    if ((threadIdx.x & 31) == 0 && (threadIdx.x >> 5) < issuers) {
        u64 pol;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
        const u32 sd = (u32)__cvta_generic_to_shared(s_d), stt = (u32)__cvta_generic_to_shared(s_t);
        const int64_t nbatch = (nchunks + batch - 1) / batch;
        for (;;) {
            const int64_t bt = (int64_t)atomicAdd(&state[0], 1u);
            if (bt >= nbatch) break;
            const int64_t c0 = bt * batch, c1 = c0 + batch < nchunks ? c0 + batch : nchunks;
            for (int64_t c = c0; c < c1; c++) {
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
                             :: "l"(dist + c * per), "r"(sd), "r"(chunk), "l"(pol) : "memory");
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
                             :: "l"(tri + c * per), "r"(stt), "r"(chunk), "l"(pol) : "memory");
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                // at most DEPTH + 1 chunk pairs in flight per issuing lane
                asm volatile("cp.async.bulk.wait_group %0;" :: "n"(DEPTH) : "memory");
            }
        }
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }
}

struct CellOut { float d; int t; };

// A cell within fp32 noise of the surface (finish_cell): the triangle closest to X among t, its three edge neighbours and
// the fan around its corner nearest to X (at most 32 of it) is found in fp64, and distance, sign and id are taken from it.
// A distance that fp64 cannot tell from zero (a cell centre on a vertex, an edge, a face: |n . r| of an in-plane r is
// rounding noise of ~1e-16 |r|) is zero, and a zero has no sign -- not -1e-17 or +1e-17 by the luck of the rounding.
// A few hundred cells per million come here: the emit kernel collects them and works them off in a loop of its own at the
// end (inlined into the sign pass, or called out of line, this code cost the whole kernel 6-17 % of its speed).
__device__ __forceinline__ CellOut near_surface_cell(const float *__restrict__ soup, const float *__restrict__ fn,
                                                  const int *__restrict__ adj, const int *__restrict__ cvid,
                                                  const int *__restrict__ perm, const VertexRec *__restrict__ vrec, int t, int xt,
                                                  double x, double y, double z, double dband) {
    const V3<double> X = mk<double>(x, y, z);
    int tb = t, kc = 0, rg = 0;
    double D = 0.0, scale = 0.0, best = 1e300;
    for (int c = 0; c < 3; c++) {
        const V3<double> dv = X - ld3d(soup + 9 * (size_t)t + 3 * c);
        const double q2 = dot(dv, dv);
        if (q2 < best) { best = q2; kc = c; }
    }
    V3<double> R = X, Q = X, Nn = X;
    int he = 3 * t + (kc + 2) % 3;                           // the half-edge of t that arrives at the corner
    // one loop, one instance of the fp64 point-triangle routine: candidate 0 is t, 1..3 its edge neighbours, then the fan
    for (int c = 0; c < 36; c++) {
        int tt = t;
        if (c >= 1 && c <= 3) {
            const int tw = adj[3 * (size_t)t + (c - 1)];
            if (tw < 0 || tw / 3 == t) continue;
            tt = tw / 3;
        } else if (c > 3) {
            // the fan matters only where the cell is as close to the corner as to the surface (within the same noise):
            // elsewhere the closest point lies in a face or on an edge, and the edge neighbours were all there is to ask
            if (c == 4) {
                const double lim = D + 1e-5 * scale;
                if (best > lim * lim) break;
            }
            const int tw = adj[he];                          // its twin leaves the corner in the next triangle of the fan
            if (tw < 0 || tw / 3 == t) break;
            tt = tw / 3;
            he = 3 * tt + ((tw - 3 * tt) + 2) % 3;
        }
        const float *TT = soup + 9 * (size_t)tt;
        const V3<double> A2 = ld3d(TT), E0 = ld3d(TT + 3) - A2, EC = ld3d(TT + 6) - A2, R2 = X - A2;
        V3<double> n2 = cross(E0, EC), q2;
        n2 = (1.0 / sqrt(dot(n2, n2))) * n2;
        int rg2;
        const double D2 = tri_closest<double>(R2, E0, EC, n2, rg2, q2);
        if (c == 0 || D2 < D) {
            D = D2; tb = tt; rg = rg2; R = R2; Q = q2; Nn = n2;
            scale = fabs(R2.x) + fabs(R2.y) + fabs(R2.z) + fabs(E0.x) + fabs(E0.y) + fabs(E0.z) + fabs(EC.x) + fabs(EC.y) + fabs(EC.z);
        }
    }
    CellOut o;
    o.d = INFINITY; o.t = -1;
    if (!(D < dband)) return o;
    if (D <= 4e-15 * scale) D = 0.0;
    V3<double> PN;
    if (rg == RG_FACE) PN = Nn;
    else if (rg <= RG_E2) PN = ld3d(fn + 3 * (size_t)tb) + ld3d(fn + 3 * (size_t)(adj[3 * (size_t)tb + (rg - RG_E0)] / 3));
    else PN = ld3d(vrec[cvid[3 * (size_t)tb + (rg - RG_V0)]].axis);
    const bool neg = dot(PN, R - Q) < 0.0;
    const float d = (float)D;
    o.d = (neg && d != 0.0f) ? -d : d;
    o.t = tb == t ? xt : perm[tb];
    return o;
}

// Populated cell: band decision (fp64 re-check near the band edge) and the sign from the
// pseudonormal of the closest feature of the winning triangle.
__device__ __forceinline__ CellOut finish_cell(const MeshView &mv, const GridParams &g, int i, int j, int k, u64 pack,
                                               u32 &recheck, bool &near_surface) {
    CellOut o;
    o.d = INFINITY; o.t = -1;
    float d = __uint_as_float((u32)(pack >> 32));
    const int xt = (int)((u32)pack >> 2);          // the caller's id of the winning triangle
    if (((u32)pack & FL_SURE) && d < g.band - g.guard) {
        // the winning extrusion already told the side and the band test is clear
        o.d = (((u32)pack & FL_NEG) && d != 0.0f) ? -d : d;
        o.t = xt;
        return o;
    }
    const int t = mv.inv_perm[xt];
    const float *T = mv.soup + 9 * (size_t)t, *N = mv.fn + 3 * (size_t)t;
    bool redo = !(d < g.band - g.guard);
    f3 a = ld3(T), e0 = ld3(T + 3) - a, ec = ld3(T + 6) - a, n = ld3(N);
    f3 x = mk<float>(fmaf((float)i, g.h, g.ox), fmaf((float)j, g.h, g.oy), fmaf((float)k, g.h, g.oz));
    int rg; f3 q;
    tri_closest<float>(x - a, e0, ec, n, rg, q);
    f3 pn;
    if (rg == RG_FACE) pn = n;
    else if (rg <= RG_E2) pn = n + ld3(mv.fn + 3 * (size_t)(mv.adj[3 * (size_t)t + (rg - RG_E0)] / 3));
    else pn = ld3(mv.vrec[mv.cvid[3 * (size_t)t + (rg - RG_V0)]].axis);
    f3 dv = (x - a) - q;
    float s = dot(pn, dv);
    bool neg = s < 0.0f;
    if (fabsf(s) <= 1e-3f * sqrtf(dot(pn, pn) * dot(dv, dv)) || tiny_vs(g, d, x - a)) redo = true;
    if (redo) {
        // fp64 on the same winning triangle: exact cell position, distance, region, sign
        recheck++;
        V3<double> A = ld3d(T), E0 = ld3d(T + 3) - A, EC = ld3d(T + 6) - A;
        V3<double> Nn = cross(E0, EC);
        Nn = (1.0 / sqrt(dot(Nn, Nn))) * Nn;
        V3<double> X = mk<double>(g.dox + i * g.dh, g.doy + j * g.dh, g.doz + k * g.dh);
        V3<double> Q;
        double D = tri_closest<double>(X - A, E0, EC, Nn, rg, Q);
        const V3<double> R = X - A;
        const double scale = fabs(R.x) + fabs(R.y) + fabs(R.z) + fabs(E0.x) + fabs(E0.y) + fabs(E0.z) + fabs(EC.x) + fabs(EC.y) + fabs(EC.z);
        if (D <= 1e-5 * scale) {
            // Within fp32 noise of the surface the fp32 minimum may belong to a NEIGHBOUR of the closest triangle (3e-8
            // beside 9e-9: the order of two such candidates is rounding luck), and beside a sharp edge the neighbour's side
            // of the surface is the other one: the triangles around the winner are measured in fp64 too, the closest decides
            // (a few hundred cells per million: the caller hands them to near_surface_cell)
            near_surface = true;
            return o;
        }
        if (!(D < g.dband)) return o;                         // strictly inside the band
        V3<double> PN;
        if (rg == RG_FACE) PN = Nn;
        else if (rg <= RG_E2) PN = ld3d(N) + ld3d(mv.fn + 3 * (size_t)(mv.adj[3 * (size_t)t + (rg - RG_E0)] / 3));
        else PN = ld3d(mv.vrec[mv.cvid[3 * (size_t)t + (rg - RG_V0)]].axis);
        neg = dot(PN, (X - A) - Q) < 0.0;
        d = (float)D;
    }
    o.d = (neg && d != 0.0f) ? -d : d;
    o.t = xt;
    return o;
}

// One WARP per active brick (8x8x8 cells, 4 KiB of packed scratch), four rounds of 128 cells; a lane takes four cells per
// round (half of an 8-cell row segment = one 32-B sector of each grid); all eight 16-byte loads of a lane are issued up
// front.  A cell whose winning extrusion already told the side and whose band test is clear is unpacked on the spot,
// branch-free (an empty cell's distance bits are a NaN and fail the band test by themselves).  The others -- about one
// populated cell in a hundred: the eps / smooth-feature margins of the prisms, wedge end caps, the band edge -- are noted in a
// queue in shared memory and worked off 32 at a time after the four rounds, at ONE call site of the large, divergent
// sign pass.  Only row segments that hold a populated cell are written: the sentinel fill has been there before.  No
// block-wide rendezvous.  (A block per brick with a queue per warp: 325 M warp instructions and 0.43 ms at C5; this: 183 M, 0.35 ms.)
// SPARSE: the brick goes out whole (sentinels included) at its slot of a band-sparse output, [slot][512] cells in the
// scratch's own order (k&7, j&7, i&7; x fastest) -- sdf_compute_sparse; no dense grid, no sentinel fill.
#define EB_BT 128
#define EB_WARPS (EB_BT / 32)
template <bool SPARSE>
__global__ void __launch_bounds__(EB_BT, 8) emit_bricks_kernel(MeshView mv, GridParams g, const int *__restrict__ list,
                                                            int nslots, const u64 *__restrict__ scratch,
                                                            float *__restrict__ dist, int *__restrict__ tri,
                                                            u64 *__restrict__ ctr) {
    __shared__ unsigned short s_cell[EB_WARPS][BRICK_CELLS];       // the warp's queue: cells whose sign is still open
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int slot = blockIdx.x * EB_WARPS + w;
    if (slot >= nslots) return;
    const int b = list[slot];
    const int bx = b % g.nbx, by = (b / g.nbx) % g.nby, bz = b / (g.nbx * g.nby);
    u32 band = 0, recheck = 0;
    const float clear = g.band - g.guard;
    const ulonglong2 *src = (const ulonglong2 *)(scratch + (size_t)slot * BRICK_CELLS) + 2 * lane;
    // all eight loads of the lane in flight before the first is used
    ulonglong2 ld[8];
#pragma unroll
    for (int r = 0; r < 4; r++) { ld[2 * r] = __ldcs(src + 64 * r); ld[2 * r + 1] = __ldcs(src + 64 * r + 1); }
    int n = 0;                                                 // entries in the warp's queue (same value in every lane)
    // cell c0 = 128 r + 4 lane: x = (4 lane) & 7, y = (lane >> 1) & 7, z = 2 r + (lane >> 4)
    const int i = bx * 8 + ((4 * lane) & 7), j = by * 8 + ((lane >> 1) & 7);
    const size_t o_row = (size_t)j * g.nx + i, o_slice = (size_t)g.ny * g.nx;
    const bool row_ok = j < g.ny, vec_ok = g.vec4 && i + 3 < g.nx;
#pragma unroll
    for (int r = 0; r < 4; r++) {
        const u64 p[4] = {ld[2 * r].x, ld[2 * r].y, ld[2 * r + 1].x, ld[2 * r + 1].y};
        // two z-slices without a candidate (a band sheet rarely crosses all eight slices of a brick): nothing to unpack or write
        if (__all_sync(0xffffffffu, (u32)((p[0] & p[1] & p[2] & p[3]) >> 32) == 0xFFFFFFFFu)) {
            if (!SPARSE) continue;
        }
        const int c0 = 128 * r + 4 * lane;
        float od[4];
        int ot[4];
        bool any = false;
        u32 nq = 0;                                            // this lane's cells for the queue (bit c)
#pragma unroll
        for (int c = 0; c < 4; c++) {
            // an empty cell holds all ones: its distance bits are a NaN and fail `d < clear` by themselves
            const u32 hi = (u32)(p[c] >> 32), lo = (u32)p[c];
            const float d = __uint_as_float(hi);
            const bool sure = (lo & FL_SURE) && d < clear;     // the winning extrusion already told the side, band test clear
            od[c] = sure ? (((lo & FL_NEG) && d != 0.0f) ? -d : d) : INFINITY;
            ot[c] = sure ? (int)(lo >> 2) : -1;
            any |= sure;
            band += sure ? 1u : 0u;
            if (!sure && hi != 0xFFFFFFFFu) nq |= 1u << c;
        }
        if (__any_sync(0xffffffffu, nq != 0u)) {
            // (rare: about one cell in a hundred) queue positions = exclusive prefix of the lanes' counts
            const int mine = __popc(nq);
            int inc = mine;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += v;
            }
            const int total = __shfl_sync(0xffffffffu, inc, 31);
            int q = n + inc - mine;
#pragma unroll
            for (int c = 0; c < 4; c++)
                if (nq & (1u << c)) { s_cell[w][q] = (unsigned short)(c0 + c); q++; }
            n += total;
        }
        // the two halves of a row segment go out together (full 32-B sectors)
        const bool other = __shfl_xor_sync(0xffffffffu, any ? 1 : 0, 1) != 0;     // (every lane takes part: no short circuit)
        const bool seg = any || other;
        const int k = bz * 8 + 2 * r + (lane >> 4);
        if (SPARSE) {
            const size_t o = (size_t)slot * BRICK_CELLS + c0;
            *(float4 *)(dist + o) = make_float4(od[0], od[1], od[2], od[3]);
            *(int4 *)(tri + o) = make_int4(ot[0], ot[1], ot[2], ot[3]);
        } else if (seg && row_ok && k < g.nz) {
            const size_t o = (size_t)k * o_slice + o_row;
            if (vec_ok) {
                *(float4 *)(dist + o) = make_float4(od[0], od[1], od[2], od[3]);
                *(int4 *)(tri + o) = make_int4(ot[0], ot[1], ot[2], ot[3]);
            } else {
#pragma unroll
                for (int c = 0; c < 4; c++)
                    if (i + c < g.nx && ot[c] >= 0) { dist[o + c] = od[c]; tri[o + c] = ot[c]; }
            }
        }
    }
    // the sign pass proper, 32 queued cells at a time (one call site: finish_cell is large).  The packed value is read
    // again from the scratch (an L2 hit); the single-cell stores come after the warp's segment stores above.
    __syncwarp();
    int n2 = 0;                                                // cells within fp32 noise of the surface: a second, colder queue
    for (int q0 = 0; q0 < n; q0 += 32) {
        bool near = false;
        int c = 0;
        if (q0 + lane < n) {
            c = s_cell[w][q0 + lane];
            const int ci = bx * 8 + (c & 7), cj = by * 8 + ((c >> 3) & 7), ck = bz * 8 + (c >> 6);
            const CellOut o = finish_cell(mv, g, ci, cj, ck, __ldcg(scratch + (size_t)slot * BRICK_CELLS + c), recheck, near);
            if (o.t >= 0) {
                const size_t idx = SPARSE ? (size_t)slot * BRICK_CELLS + c : ((size_t)ck * g.ny + cj) * g.nx + ci;
                dist[idx] = o.d; tri[idx] = o.t;
                band++;
            }
        }
        const unsigned nm = __ballot_sync(0xffffffffu, near);
        if (nm) {
            // (the slots written here were read above: entry n2 + rank <= q0 + lane)
            __syncwarp();
            if (near) s_cell[w][n2 + __popc(nm & ((1u << lane) - 1u))] = (unsigned short)c;
            n2 += __popc(nm);
            __syncwarp();
        }
    }
    for (int q0 = 0; q0 < n2; q0 += 32) {
        if (q0 + lane < n2) {
            const int c = s_cell[w][q0 + lane];
            const int ci = bx * 8 + (c & 7), cj = by * 8 + ((c >> 3) & 7), ck = bz * 8 + (c >> 6);
            const u64 pack = __ldcg(scratch + (size_t)slot * BRICK_CELLS + c);
            const int xt = (int)((u32)pack >> 2);
            const CellOut o = near_surface_cell(mv.soup, mv.fn, mv.adj, mv.cvid, mv.perm, mv.vrec, mv.inv_perm[xt], xt,
                                                g.dox + ci * g.dh, g.doy + cj * g.dh, g.doz + ck * g.dh, g.dband);
            if (o.t >= 0) {
                const size_t idx = SPARSE ? (size_t)slot * BRICK_CELLS + c : ((size_t)ck * g.ny + cj) * g.nx + ci;
                dist[idx] = o.d; tri[idx] = o.t;
                band++;
            }
        }
    }
    // statistics: warp sums into counters spread over CTR_SLOTS lines (same-address atomics serialise in L2)
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        band += __shfl_xor_sync(0xffffffffu, band, o);
        recheck += __shfl_xor_sync(0xffffffffu, recheck, o);
    }
    if (lane == 0) {
        u64 *sp = ctr + CTR_SPREAD + (slot & (CTR_SLOTS - 1)) * 8;
        if (band) atomicAdd(sp + SP_BAND, (u64)band);
        if (recheck) atomicAdd(sp + SP_RECHECK, (u64)recheck);
    }
}

// ---------------------------------------------------------------------------------------
// host driver
// ---------------------------------------------------------------------------------------
template <typename T>
static int ensure(sdf_mesh *m, T **p, size_t *cap, size_t need, cudaStream_t st) {
    if (*cap >= need && *p) return SDF_OK;
    if (*p) { dev_free(&m->alloc, *p, st); *p = nullptr; *cap = 0; }
    size_t want = need + need / 8 + 256;
    CKS(dev_alloc(&m->alloc, (void **)p, want * sizeof(T), st));
    *cap = want;
    return SDF_OK;
}

// A8a: the sentinel fill depends on nothing but the output pointers.  Forked onto the side stream it
// streams to HBM underneath whatever runs on `st` next: A5-A7 inside sdf_compute, or -- when
// sdf_transform starts it first -- the whole feature construction A0-A4 as well.
static int fork_sentinel_fill(sdf_mesh *m, const GridParams &g, float *dist, int *tri, cudaStream_t st, bool fork) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int64_t N = (int64_t)g.nx * g.ny * g.nz;
    const int vec = (((uintptr_t)dist & 15) == 0) && (((uintptr_t)tri & 15) == 0);
    static_assert(FILL_STATE_WORDS == 1024, "fill_state is carved out of slab_f with 1024 words (features.cu)");
    auto launch_fill = [&](cudaStream_t fs) -> int {
        stage_mark(m, SDF_T_FILL, 0, fs);
        if (vec && g.fill_mode != 1) {
            const int iss = g.fill_issuers | (g.fill_sm_share << 8) | (g.fill_chunk_log2 << 16);
            const int chunk = 1 << g.fill_chunk_log2;
            CK(cudaMemsetAsync(m->fill_state, 0, sizeof(u32) * FILL_STATE_WORDS, fs));
            const unsigned nb = (unsigned)(sms * g.fill_ctas);
            // batch of chunks per fetch: 1 MiB per array on large grids, smaller when the grid has
            // fewer than ~8 batches per issuing lane
            int64_t bq = (N / (chunk / 4)) / ((int64_t)sms * g.fill_issuers * 8);
            const int batch = (int)(bq < 1 ? 1 : (bq > FILL_BATCH_BYTES / chunk ? FILL_BATCH_BYTES / chunk : bq));
            KL;
            switch (g.fill_depth) {
            case 0: fill_tma_kernel<0><<<nb, FILL_TMA_BT, 0, fs>>>(dist, tri, N, iss, batch, m->fill_state, 0x7F800000u, 0xFFFFFFFFu); break;
            case 1: fill_tma_kernel<1><<<nb, FILL_TMA_BT, 0, fs>>>(dist, tri, N, iss, batch, m->fill_state, 0x7F800000u, 0xFFFFFFFFu); break;
            case 2: fill_tma_kernel<2><<<nb, FILL_TMA_BT, 0, fs>>>(dist, tri, N, iss, batch, m->fill_state, 0x7F800000u, 0xFFFFFFFFu); break;
            case 4: fill_tma_kernel<4><<<nb, FILL_TMA_BT, 0, fs>>>(dist, tri, N, iss, batch, m->fill_state, 0x7F800000u, 0xFFFFFFFFu); break;
            default: fill_tma_kernel<8><<<nb, FILL_TMA_BT, 0, fs>>>(dist, tri, N, iss, batch, m->fill_state, 0x7F800000u, 0xFFFFFFFFu); break;
            }
        } else {
            int64_t fb = (N / 4 + (int64_t)FILL_BT * FILL_UNROLL - 1) / ((int64_t)FILL_BT * FILL_UNROLL);
            if (fb > (int64_t)sms * 2) fb = (int64_t)sms * 2;
            if (fb < 1) fb = 1;
            KL; fill_kernel<<<(unsigned)fb, FILL_BT, 0, fs>>>(dist, tri, N, vec);
        }
        stage_mark(m, SDF_T_FILL, 1, fs);
        return SDF_OK;
    };
    if (!fork) return launch_fill(st);
    if (!m->side) {
        // one library-owned side stream per process (creating a stream per handle cost ~30 us
        // per sdf_compute on a fresh handle); highest priority: the few, tiny fill CTAs are
        // placed before the evaluate blocks
        static cudaStream_t g_side = nullptr;
        static int g_side_prio = -1, g_side_dev = -1;
        if (!g_side || g_side_prio != g.fill_prio || g_side_dev != dev) {
            int plo = 0, phi = 0;
            cudaDeviceGetStreamPriorityRange(&plo, &phi);
            CK(cudaStreamCreateWithPriority(&g_side, cudaStreamNonBlocking, g.fill_prio ? phi : plo));
            g_side_prio = g.fill_prio;
            g_side_dev = dev;
        }
        m->side = g_side;
    }
    CKS(ev_get(m, &m->ev_ffork));
    CKS(ev_get(m, &m->ev_fjoin));
    CK(cudaEventRecord(m->ev_ffork, st));
    CK(cudaStreamWaitEvent(m->side, m->ev_ffork, 0));
    CKS(launch_fill(m->side));
    CK(cudaEventRecord(m->ev_fjoin, m->side));
    return SDF_OK;
}

// sdf_transform: start the sentinel fill of the outputs before the feature tables exist
int start_prefill(sdf_mesh *m, const GridParams &g, float *dist, int *tri, cudaStream_t st) {
    m->ev_set[SDF_T_FILL] = false;
    return fork_sentinel_fill(m, g, dist, tri, st, true);
}

// stage boundary `point` of build_features: start the pending fill if this is where it was asked for
int maybe_prefill(sdf_mesh *m, int point, cudaStream_t st) {
    if (!m->pre_g || m->pre_at != point) return SDF_OK;
    const GridParams *g = m->pre_g;
    m->pre_g = nullptr;
    return start_prefill(m, *g, m->pre_dist, m->pre_tri, st);
}

static MeshView make_view(const sdf_mesh *m) {
    MeshView mv;
    mv.soup = m->soup; mv.fn = m->fn; mv.fsm = m->fsm; mv.erec = m->erec; mv.vrec = m->vrec; mv.vmint = m->vmint;
    mv.cone_list = m->cone_list; mv.vsm = m->vsm;
    mv.cvid = m->cvid; mv.adj = m->adj; mv.perm = m->perm; mv.inv_perm = m->inv_perm;
    mv.F = (int)m->F; mv.E = (int)m->Elive; mv.V = (int)m->V; mv.NC = (int)m->NC;
    mv.P = m->F + m->Elive + m->NC;
    return mv;
}

// A6a workspace: brick flags / table / list, scan partials, big-polyhedron list -- one slab, grown on demand,
// taken in the order of stream `as`
static int alloc_brick_ws(sdf_mesh *m, const GridParams &g, cudaStream_t as) {
    const int64_t P = m->F + m->E + 2 * m->V;
    const int64_t nbricks = (int64_t)g.nbx * g.nby * g.nbz;
    for (int pass = 0; pass < 2; pass++) {
        Carver c(pass ? m->slab_ws : nullptr);
        m->brick_flag = c.take<unsigned char>((size_t)nbricks);
        m->brick_table = c.take<int>((size_t)nbricks);
        m->brick_list = c.take<int>((size_t)nbricks);
        m->scan_ws = c.take<u64>(scan_ws_elems(nbricks));
        m->big_list = c.take<u32>((size_t)P);
        if (pass == 0 && (c.off > m->slab_ws_cap || !m->slab_ws)) {
            if (m->slab_ws) { dev_free(&m->alloc, m->slab_ws, as); m->slab_ws = nullptr; m->slab_ws_cap = 0; }
            const size_t want = c.off + c.off / 8 + 256;
            CKS(dev_alloc(&m->alloc, &m->slab_ws, want, as));
            m->slab_ws_cap = want;
        }
    }
    return SDF_OK;
}

// A6a on stream `ps` (workspace already carved): reset the flags and the per-compute counters; mark the bricks the band
// can reach (unless a kernel of sdf_create did: `marked`); prefix sum -> brick table, list and the total in
// d_ctr[CTR_BRICKS].  Needs the soup, the face normals and V; sdf_transform runs it beside the edge stage.
static int reset_bricks(sdf_mesh *m, const GridParams &g, cudaStream_t ps) {
    const int64_t nbricks = (int64_t)g.nbx * g.nby * g.nbz;
    m->ev_set[SDF_T_CLIP_SCAN] = false;
    CK(cudaMemsetAsync(m->brick_flag, 0, (size_t)nbricks, ps));
    CK(cudaMemsetAsync(m->d_ctr + CTR_POLY, 0, sizeof(u64) * (CTR_TOTAL - CTR_POLY), ps));
    return SDF_OK;
}
static int scan_bricks(sdf_mesh *m, const GridParams &g, cudaStream_t ps, bool marked) {
    const int64_t nbricks = (int64_t)g.nbx * g.nby * g.nbz;
    stage_mark(m, SDF_T_CLIP_SCAN, 0, ps);
    if (!marked) {
        const MeshView mv = make_view(m);
        if (mv.F >= (1 << 21)) { KL; brick_mark_kernel<false><<<(unsigned)((mv.F + 255) / 256), 256, 0, ps>>>(mv, g, m->brick_flag); }
        else { KL; brick_mark_kernel<true><<<(unsigned)((4 * (int64_t)mv.F + 255) / 256), 256, 0, ps>>>(mv, g, m->brick_flag); }
    }
    CKS(launch_scan(BrickIn{m->brick_flag}, BrickOut{m->brick_table, m->brick_list}, nbricks, m->scan_ws, m->d_ctr + CTR_BRICKS, ps));
    CK(cudaGetLastError());
    return SDF_OK;
}

// sdf_transform, before build_features forks the vertex stream (tile builder: the marking kernel runs later)
int maybe_alloc_brick_ws(sdf_mesh *m, cudaStream_t st) {
    if (!m->hoist_g) return SDF_OK;
    return alloc_brick_ws(m, *m->hoist_g, st);          // (the resets go with the marking kernel: maybe_prepare_bricks)
}

// sdf_transform, global builder: workspace + reset on `st`, and a device copy of the grid for tri_geom_kernel, which
// marks the bricks itself
int maybe_begin_bricks(sdf_mesh *m, cudaStream_t st, const GridParams **g_dev, unsigned char **flag) {
    *g_dev = nullptr; *flag = nullptr;
    if (!m->hoist_g) return SDF_OK;
    CKS(alloc_brick_ws(m, *m->hoist_g, st));
    CKS(reset_bricks(m, *m->hoist_g, st));
    CK(cudaMemcpyAsync(m->hoist_g_dev, m->hoist_g, sizeof(GridParams), cudaMemcpyHostToDevice, st));
    *g_dev = m->hoist_g_dev;
    *flag = m->brick_flag;
    return SDF_OK;
}

// sdf_transform: stage boundary of build_features after the vertex kernels (stream vs, forked from st)
int maybe_prepare_bricks(sdf_mesh *m, cudaStream_t st, cudaStream_t vs, bool marked) {
    if (!m->hoist_g) return SDF_OK;
    const GridParams *g = m->hoist_g;
    m->hoist_g = nullptr;
    (void)st;
    if (!marked) CKS(reset_bricks(m, *g, vs));          // off the caller's stream: two fewer operations in front of the edge stage
    CKS(scan_bricks(m, *g, vs, marked));
    stage_mark(m, SDF_T_CLIP_SCAN, 1, vs);
    m->bricks_ready = true;        // the total travels with the validation flags (the host crossing)
    return SDF_OK;
}

int run_compute(sdf_mesh *m, const GridParams &g_in, float *dist, int *tri, cudaStream_t st, bool prefilled, SparseOut *sp) {
    GridParams g = g_in;
    {
        // a mesh with few polyhedra cannot fill the GPU with one lane per polyhedron: hand more
        // of them to the block-per-polyhedron kernel
        const int64_t P0 = m->F + m->Elive + m->NC;
        g.big_rows = P0 < 4096 ? 8 : (P0 < 65536 ? 64 : (int)BIG_ROWS);
        g.big_ni = P0 < 4096 ? 4 : (P0 < 65536 ? 16 : BIG_NI);
    }
    const MeshView mv = make_view(m);
    const int64_t P = mv.P;
    const int64_t nbricks = (int64_t)g.nbx * g.nby * g.nbz;
    const bool hoisted = m->bricks_ready;
    m->bricks_ready = false;

    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    for (int i = SDF_T_CLEAR; i < SDF_T_COUNT; i++)
        if (!(prefilled && i == SDF_T_FILL)) m->ev_set[i] = false;
    // the fill is forked here (or, fill_mode 4, after the host crossing below) unless sdf_transform
    // already started it ahead of the feature construction
    if (sp) g.fill_mode = 5;                       // band-sparse output: no dense grid to fill
    const bool forked = !sp && (prefilled || g.fill_mode < 2 || g.fill_mode == 4);
    auto fork_fill = [&]() -> int { return fork_sentinel_fill(m, g, dist, tri, st, true); };
    auto launch_fill = [&](cudaStream_t fs) -> int { return fork_sentinel_fill(m, g, dist, tri, fs, false); };
    if (prefilled) {}
    else if (g.fill_mode < 2) CKS(fork_fill());
    else if (g.fill_mode == 3) CKS(launch_fill(st));

    // A6a: brick table and its total (host crossing: the total sizes the launch and the scratch), unless
    // sdf_transform already ran it beside the edge stage and fetched the total with the validation flags
    u64 bricks = 0;
    if (hoisted) {
        bricks = m->h_ctr[CTR_BRICKS];
    } else {
        CKS(alloc_brick_ws(m, g, st));
        CKS(reset_bricks(m, g, st));
        CKS(scan_bricks(m, g, st, false));
        CK(cudaMemcpyAsync(&bricks, m->d_ctr + CTR_BRICKS, sizeof(bricks), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        stage_mark(m, SDF_T_CLIP_SCAN, 1, st);
    }
    // fork the fill first: its CTAs claim their SMs while the GPU is still empty (the scratch
    // allocation and its clear come next), before the evaluate blocks flood it
    if (g.fill_mode == 4 && !prefilled) CKS(fork_fill());
    if (sp) {
        sp->count = (int64_t)bricks;
        m->h_ctr[CTR_BRICKS] = bricks;
        m->last_bricks_total = nbricks;
        m->last_stream = st;
        if ((int64_t)bricks > sp->cap) return SDF_ENOMEM;          // the caller learns the count and comes back
        dist = sp->dist; tri = sp->tri;
        if (bricks) CK(cudaMemcpyAsync(sp->ids, m->brick_list, sizeof(int) * (size_t)bricks, cudaMemcpyDeviceToDevice, st));
    }
    CKS(ensure(m, &m->scratch, &m->scratch_cap, (size_t)(bricks ? bricks : 1) * BRICK_CELLS, st));
    stage_mark(m, SDF_T_CLEAR, 0, st);
    if (bricks) CK(cudaMemsetAsync(m->scratch, 0xFF, (size_t)bricks * BRICK_CELLS * sizeof(u64), st));
    stage_mark(m, SDF_T_CLEAR, 1, st);

    // A5 + A6b + A7: clip every polyhedron, flatten the small ones per warp and evaluate them;
    // big ones one block each (dynamic fetch)
    if (bricks) {
        stage_mark(m, SDF_T_EVALUATE, 0, st);
        const int ppw = P < (1 << 17) ? 4 : (P < (1 << 20) ? 8 : 32);
        int64_t nblk = (P + (int64_t)ppw * ES_WARPS - 1) / ((int64_t)ppw * ES_WARPS);
        EvalOrder eo = {0, 0, 0, 0};
        if (g.eval_chunk > 0 && (mv.E > 0 || mv.NC > 0) && P >= (1 << 17)) {
            const int64_t nf = (mv.F + ppw - 1) / ppw, ne = ((int64_t)mv.E + ppw - 1) / ppw, nc = ((int64_t)mv.NC + ppw - 1) / ppw;
            int64_t K = (nf + ne + nc) / g.eval_chunk;
            if (K < 1) K = 1;
            eo.chunks = K;
            eo.wf = (nf + K - 1) / K; eo.we = (ne + K - 1) / K; eo.wc = (nc + K - 1) / K;
            nblk = (K * (eo.wf + eo.we + eo.wc) + ES_WARPS - 1) / ES_WARPS;
        }
        const unsigned split = P < 65536 ? EBIG_SPLIT : (P < (1 << 20) ? 2 : 1);
        if (g.cdp) {
            CKS(run_cdp_evaluate(m, mv, g, st));
        } else {
        KL;
        if (g.serial_loop) evaluate_small_kernel<true><<<(unsigned)nblk, 32 * ES_WARPS, 0, st>>>(mv, g, m->big_list, m->brick_table, m->scratch, m->d_ctr, ppw, eo);
        else evaluate_small_kernel<false><<<(unsigned)nblk, 32 * ES_WARPS, 0, st>>>(mv, g, m->big_list, m->brick_table, m->scratch, m->d_ctr, ppw, eo);
        KL; evaluate_big_kernel<<<dim3((unsigned)(sms * 4 / split), split), EBIG_BT, 0, st>>>(mv, g, m->big_list, m->brick_table, m->scratch, m->d_ctr);
        }
        stage_mark(m, SDF_T_EVALUATE, 1, st);
    }
    // A8b: join the fill, then overwrite the active bricks
    if (forked) CK(cudaStreamWaitEvent(st, m->ev_fjoin, 0));
    else if (g.fill_mode == 2) CKS(launch_fill(st));
    if (bricks) {
        stage_mark(m, SDF_T_EMIT, 0, st);
        KL;
        const unsigned eb = (unsigned)((bricks + EB_WARPS - 1) / EB_WARPS);
        if (sp) emit_bricks_kernel<true><<<eb, EB_BT, 0, st>>>(mv, g, m->brick_list, (int)bricks, m->scratch, dist, tri, m->d_ctr);
        else emit_bricks_kernel<false><<<eb, EB_BT, 0, st>>>(mv, g, m->brick_list, (int)bricks, m->scratch, dist, tri, m->d_ctr);
        stage_mark(m, SDF_T_EMIT, 1, st);
    }
    CK(cudaGetLastError());
    m->last_stream = st;
    m->h_ctr[CTR_BRICKS] = bricks;
    m->last_bricks_total = nbricks;
    return SDF_OK;
}

// ---------------------------------------------------------------------------------------
// closest points (the closest point transform proper).
// One thread per cell: the point of the winning triangle nearest to the cell centre, +inf outside
// the band.  HBM-bound: 4 B read + 12 B written per cell; the triangle gathers stay in L2 (the band
// is walked in grid order and the soup is spatially binned).
// ---------------------------------------------------------------------------------------
// Closest point of the triangle (0, e0, ec) to r.  Not tri_closest: that one ranks the candidate edges by their
// squared distances, which is right for the distance but leaves the POINT undecided within d * sqrt(2 eps) -- far
// from the triangle a vertex and a point 1e-4 along an edge are equally far in fp32.  Here the edge whose foot point
// is interior wins outright: a point outside an edge's half-plane whose foot lies inside the segment has that foot
// as the closest point of the whole half-plane, hence of the triangle; only end points are ranked by distance.
__device__ __forceinline__ void edge_candidate(f3 r, f3 o, f3 e, float &best, bool &interior, f3 &q) {
    const f3 ro = r - o;
    float t = dot(ro, e) / dot(e, e);
    const bool in = t > 0.0f && t < 1.0f;
    t = fminf(fmaxf(t, 0.0f), 1.0f);
    const f3 c = o + t * e, d = r - c;
    const float d2 = dot(d, d);
    if ((in && !interior) || (in == interior && d2 < best)) { best = d2; q = c; interior = in; }
}
__device__ __forceinline__ f3 tri_closest_point(f3 r, f3 e0, f3 ec, f3 n) {
    const f3 e1 = ec - e0;
    const float s0 = dot(cross(n, e0), r), s1 = dot(cross(n, e1), r - e0), s2 = -dot(cross(n, ec), r - ec);
    if (s0 >= 0.0f && s1 >= 0.0f && s2 >= 0.0f) return r - dot(n, r) * n;
    float best = INFINITY;
    bool interior = false;
    f3 q = mk<float>(0.0f, 0.0f, 0.0f);
    if (s0 < 0.0f) edge_candidate(r, q, e0, best, interior, q);
    if (s1 < 0.0f) edge_candidate(r, e0, e1, best, interior, q);
    if (s2 < 0.0f) edge_candidate(r, mk<float>(0.0f, 0.0f, 0.0f), ec, best, interior, q);
    return q;
}

__device__ __forceinline__ void closest_point_of(const MeshView &mv, const GridParams &g, int xt, int64_t c, float *o) {
    o[0] = o[1] = o[2] = INFINITY;
    if (xt >= 0 && xt < mv.F) {
        const int i = (int)(c % g.nx), j = (int)((c / g.nx) % g.ny), k = (int)(c / ((int64_t)g.nx * g.ny));
        const int t = mv.inv_perm[xt];
        const float *T = mv.soup + 9 * (size_t)t;
        const f3 a = ld3(T), x = mk<float>(fmaf((float)i, g.h, g.ox), fmaf((float)j, g.h, g.oy), fmaf((float)k, g.h, g.oz));
        const f3 q = tri_closest_point(x - a, ld3(T + 3) - a, ld3(T + 6) - a, ld3(mv.fn + 3 * (size_t)t));
        o[0] = a.x + q.x; o[1] = a.y + q.y; o[2] = a.z + q.z;
    }
}

// VEC = 4: a thread takes four consecutive cells (one 128-bit load of ids, three 128-bit streaming
// stores of points); VEC = 1 for unaligned buffers and the ragged tail
template <int VEC>
__global__ void __launch_bounds__(256) closest_points_kernel(MeshView mv, GridParams g, const int *__restrict__ tri,
                                                             float *__restrict__ cp, int64_t first, int64_t n) {
    const int64_t c = first + ((int64_t)blockIdx.x * 256 + threadIdx.x) * VEC;
    if (c >= n) return;
    if (VEC == 4) {
        const int4 t4 = *(const int4 *)(tri + c);
        const int xt[4] = {t4.x, t4.y, t4.z, t4.w};
        float o[12];
        if ((xt[0] & xt[1] & xt[2] & xt[3]) < 0 && xt[0] < 0 && xt[1] < 0 && xt[2] < 0 && xt[3] < 0) {
#pragma unroll
            for (int u = 0; u < 12; u++) o[u] = INFINITY;
        } else {
#pragma unroll
            for (int u = 0; u < 4; u++) closest_point_of(mv, g, xt[u], c + u, o + 3 * u);
        }
        float4 *dst = (float4 *)(cp + 3 * c);
        __stcs(dst, make_float4(o[0], o[1], o[2], o[3]));
        __stcs(dst + 1, make_float4(o[4], o[5], o[6], o[7]));
        __stcs(dst + 2, make_float4(o[8], o[9], o[10], o[11]));
    } else {
        float o[3];
        closest_point_of(mv, g, tri[c], c, o);
        cp[3 * c] = o[0]; cp[3 * c + 1] = o[1]; cp[3 * c + 2] = o[2];
    }
}

// After a TMA fill of the whole output with +inf: only the cells of the band are visited for real.
// A block streams CPS_LOADS * 256 int4 of ids (all loads issued before any is looked at) and queues the
// band cells it meets (0.5 % of a grid, in clusters) in shared memory; the queue is then worked off a
// thread per entry, so the expensive part -- gathers and the seven-region routine -- runs on full warps
// instead of on the odd lane of a streaming warp.
#define CPS_LOADS 4
#define CPS_CELLS (256 * CPS_LOADS * 4)
__global__ void __launch_bounds__(256) closest_points_sparse_kernel(MeshView mv, GridParams g, const int *__restrict__ tri,
                                                                    float *__restrict__ cp, int64_t n4) {
    __shared__ int s_n;
    __shared__ unsigned short s_cell[CPS_CELLS];       // cell index within the block's range
    __shared__ int s_tri[CPS_CELLS];
    if (threadIdx.x == 0) s_n = 0;
    const int64_t qb = (int64_t)blockIdx.x * (256 * CPS_LOADS);       // in units of int4
    const int64_t nq = n4 >> 2;
    int4 t4[CPS_LOADS];
#pragma unroll
    for (int u = 0; u < CPS_LOADS; u++) {
        const int64_t q = qb + u * 256 + threadIdx.x;
        t4[u] = q < nq ? __ldcs((const int4 *)tri + q) : make_int4(-1, -1, -1, -1);
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < CPS_LOADS; u++) {
        const int xt[4] = {t4[u].x, t4[u].y, t4[u].z, t4[u].w};
        if ((xt[0] & xt[1] & xt[2] & xt[3]) < 0) continue;            // all four negative: no band cell
#pragma unroll
        for (int e = 0; e < 4; e++)
            if (xt[e] >= 0) {
                const int k = atomicAdd(&s_n, 1);
                s_cell[k] = (unsigned short)((u * 256 + threadIdx.x) * 4 + e);
                s_tri[k] = xt[e];
            }
    }
    __syncthreads();
    const int nk = s_n;
    for (int k = threadIdx.x; k < nk; k += 256) {
        const int64_t c = qb * 4 + s_cell[k];
        float o[3];
        closest_point_of(mv, g, s_tri[k], c, o);
        cp[3 * c] = o[0]; cp[3 * c + 1] = o[1]; cp[3 * c + 2] = o[2];
    }
}

int run_closest_points(sdf_mesh *m, const GridParams &g, const int *tri, float *cp, cudaStream_t st) {
    const MeshView mv = make_view(m);
    const int64_t n = (int64_t)g.nx * g.ny * g.nz;
    const bool vec = (((uintptr_t)tri & 15) == 0) && (((uintptr_t)cp & 15) == 0);
    if (vec && n % 8 == 0 && n >= (1 << 20) && !g.plain_cpt) {
        // large aligned grids: +inf over everything with TMA bulk stores (the two halves of cp play
        // the two arrays of the sentinel fill), then the band only
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (!m->cp_state) CKS(dev_alloc(&m->alloc, (void **)&m->cp_state, sizeof(u32) * FILL_STATE_WORDS, st));
        CK(cudaMemsetAsync(m->cp_state, 0, sizeof(u32) * FILL_STATE_WORDS, st));
        const int64_t half = 3 * n / 2;
        const int chunk = 1 << g.fill_chunk_log2;
        int64_t bq = (half / (chunk / 4)) / ((int64_t)sms * g.fill_issuers * 8);
        const int batch = (int)(bq < 1 ? 1 : (bq > FILL_BATCH_BYTES / chunk ? FILL_BATCH_BYTES / chunk : bq));
        KL; fill_tma_kernel<2><<<(unsigned)(sms * 4), FILL_TMA_BT, 0, st>>>(cp, (int *)(cp + half), half,
                                                                         g.fill_issuers | (8 << 8) | (g.fill_chunk_log2 << 16), batch,
                                                                         m->cp_state, 0x7F800000u, 0x7F800000u);
        KL; closest_points_sparse_kernel<<<(unsigned)((n / 4 + 256 * CPS_LOADS - 1) / (256 * CPS_LOADS)), 256, 0, st>>>(mv, g, tri, cp, n);
        CK(cudaGetLastError());
        m->last_stream = st;
        return SDF_OK;
    }
    const int64_t n4 = vec ? (n & ~(int64_t)3) : 0;
    if (n4) { KL; closest_points_kernel<4><<<(unsigned)((n4 / 4 + 255) / 256), 256, 0, st>>>(mv, g, tri, cp, 0, n4); }
    if (n > n4) { KL; closest_points_kernel<1><<<(unsigned)((n - n4 + 255) / 256), 256, 0, st>>>(mv, g, tri, cp, n4, n); }
    CK(cudaGetLastError());
    m->last_stream = st;
    return SDF_OK;
}

