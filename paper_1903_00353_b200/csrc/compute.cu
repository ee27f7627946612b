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
    const float *soup, *fn;
    const EdgeRec *erec;
    const VertexRec *vrec;
    const int *vmint, *cvid, *adj;
    int F, E, V;
    int64_t P;
};

__device__ __forceinline__ void cell_range(double mn, double mx, double o, double inv_h, int n, int &lo, int &hi) {
    double l = ceil((mn - o) * inv_h - 1e-4), u = floor((mx - o) * inv_h + 1e-4);
    l = fmin(fmax(l, 0.0), (double)n);
    u = fmax(fmin(u, (double)(n - 1)), -1.0);
    lo = (int)l; hi = (int)u;
}

__global__ void __launch_bounds__(256) clip_count_kernel(MeshView mv, GridParams g, PolyHdr *__restrict__ hdr,
                                                         unsigned char *__restrict__ brick_flag) {
    int64_t p = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (p >= mv.P) return;
    float mn[3], mx[3];
    bool emit = true;
    const float rb = g.rb, eps = g.eps;
    if (p < mv.F) {
        // face slab: triangle swept by +-rb along its normal
        const float *T = mv.soup + 9 * p, *N = mv.fn + 3 * p;
#pragma unroll
        for (int i = 0; i < 3; i++) {
            float lo = fminf(T[i], fminf(T[3 + i], T[6 + i])), hi = fmaxf(T[i], fmaxf(T[3 + i], T[6 + i]));
            float ext = g.aabb_mode ? rb : rb * fabsf(N[i]);
            mn[i] = lo - ext - eps; mx[i] = hi + ext + eps;
        }
    } else if (p < (int64_t)mv.F + mv.E) {
        // edge wedge: segment swept by the arc between n1 and n2, radius rb
        const EdgeRec &r = mv.erec[p - mv.F];
        emit = (r.cls != 0) && !g.aabb_mode;
        if (emit) {
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
        int64_t q = p - mv.F - mv.E;
        const VertexRec &r = mv.vrec[q >> 1];
        int side = (int)(q & 1);
        emit = ((r.info >> side) & 1) && !g.aabb_mode && !(side == 1 && r.cos_cone <= -1.0f);
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
    PolyHdr h;
    h.i0 = h.j0 = h.k0 = 0; h.i1 = h.j1 = h.k1 = -1; h.rows = 0;
    if (emit) {
        int i0, i1, j0, j1, k0, k1;
        double ih = 1.0 / g.dh;
        cell_range(mn[0], mx[0], g.dox, ih, g.nx, i0, i1);
        cell_range(mn[1], mx[1], g.doy, ih, g.ny, j0, j1);
        cell_range(mn[2], mx[2], g.doz, ih, g.nz, k0, k1);
        if (i0 <= i1 && j0 <= j1 && k0 <= k1) {
            h.i0 = (short)i0; h.i1 = (short)i1; h.j0 = (short)j0; h.j1 = (short)j1; h.k0 = (short)k0; h.k1 = (short)k1;
            h.rows = (u32)(j1 - j0 + 1) * (u32)(k1 - k0 + 1);
            for (int bz = k0 >> 3; bz <= (k1 >> 3); bz++)
                for (int by = j0 >> 3; by <= (j1 >> 3); by++)
                    for (int bx = i0 >> 3; bx <= (i1 >> 3); bx++)
                        brick_flag[((size_t)bz * g.nby + by) * g.nbx + bx] = 1;
        }
    }
    hdr[p] = h;
}

struct RowsIn {
    const PolyHdr *hdr;
    __device__ u64 operator()(int64_t i) const { return hdr[i].rows; }
};
struct RowsOut {
    u64 *off;
    __device__ void operator()(int64_t i, u64 ex, u64) const { off[i] = ex; }
};
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
__global__ void count_nonempty_kernel(const PolyHdr *__restrict__ hdr, int64_t P, u64 *__restrict__ ctr) {
    int64_t p = (int64_t)blockIdx.x * 256 + threadIdx.x;
    int c = __syncthreads_count(p < P && hdr[p].rows > 0);
    if (threadIdx.x == 0 && c) atomicAdd(&ctr[CTR_POLY], (u64)c);
}
__global__ void set_last_offset_kernel(u64 *off, int64_t P, const u64 *total) { off[P] = *total; }

// ---------------------------------------------------------------------------------------
// A7: flat (polyhedron, row) work items -> cells -> packed atomicMin
// ---------------------------------------------------------------------------------------
#define EV_BT 256
#define EV_IPB 1024      // work items per block
#define EV_CH 128        // polyhedra staged in shared memory per chunk

struct __align__(16) Geo {
    float f[12];
    int id, type, pad0, pad1;
};

__device__ __forceinline__ void put_min(const GridParams &g, const int *__restrict__ table, u64 *__restrict__ scratch,
                                        int i, int j, int k, float d, int id) {
    int slot = table[((size_t)(k >> 3) * g.nby + (j >> 3)) * g.nbx + (i >> 3)];
    u64 *cell = scratch + (size_t)slot * BRICK_CELLS + (((k & 7) * 8 + (j & 7)) * 8 + (i & 7));
    atomicMin(cell, ((u64)__float_as_uint(d) << 32) | (u32)id);
}

// restrict t in [tlo, thi] to s0 + t*gx >= lim
__device__ __forceinline__ void clip_ge(float s0, float gx, float lim, float &tlo, float &thi) {
    float num = lim - s0;
    if (gx > 0.0f) tlo = fmaxf(tlo, num / gx);
    else if (gx < 0.0f) thi = fminf(thi, num / gx);
    else if (num > 0.0f) thi = -1.0f;
}

__device__ __forceinline__ void process_row(const GridParams &g, const Geo &G, const PolyHdr &H, u32 row,
                                            const int *__restrict__ table, u64 *__restrict__ scratch, u32 &tested,
                                            u32 &accepted) {
    const int nj = H.j1 - H.j0 + 1;
    const int j = H.j0 + (int)(row % (u32)nj), k = H.k0 + (int)(row / (u32)nj);
    const float y = fmaf((float)j, g.h, g.oy), z = fmaf((float)k, g.h, g.oz);
    const float x0 = fmaf((float)H.i0, g.h, g.ox);
    const float reach = g.band + g.guard;          // accept d < reach; the emit pass decides exactly
    const float eps = g.eps, h = g.h;
    float tlo = 0.0f, thi = (float)(H.i1 - H.i0);
    if (G.type == 0) {
        // ---- face slab: three inward side planes through the edges + the slab
        f3 a = ld3(G.f), e0 = ld3(G.f + 3) - a, ec = ld3(G.f + 6) - a, n = ld3(G.f + 9);
        f3 e1 = ec - e0;
        f3 m0 = cross(n, e0), m1 = cross(n, e1), m2 = cross(ec, n);          // inward, |m_i| = |edge_i|
        float t0 = eps * sqrtf(dot(e0, e0)), t1 = eps * sqrtf(dot(e1, e1)), t2 = eps * sqrtf(dot(ec, ec));
        f3 r0 = mk<float>(x0 - a.x, y - a.y, z - a.z);
        if (!g.aabb_mode) {
            clip_ge(dot(m0, r0), h * m0.x, -2.0f * t0, tlo, thi);
            clip_ge(dot(m1, r0 - e0), h * m1.x, -2.0f * t1, tlo, thi);
            clip_ge(dot(m2, r0 - ec), h * m2.x, -2.0f * t2, tlo, thi);
            float dn0 = dot(n, r0), gn = h * n.x;
            clip_ge(dn0, gn, -(reach + eps), tlo, thi);
            clip_ge(-dn0, -gn, -(reach + eps), tlo, thi);
        }
        if (!(tlo <= thi)) return;
        int ia = H.i0 + (int)ceilf(tlo), ib = H.i0 + (int)floorf(thi);
        for (int i = ia; i <= ib; i++) {
            f3 r = mk<float>(fmaf((float)i, h, g.ox) - a.x, r0.y, r0.z);
            tested++;
            float d;
            if (g.aabb_mode) {
                int rg; f3 q;
                d = tri_closest<float>(r, e0, ec, n, rg, q);
            } else {
                float s0 = dot(m0, r), s1 = dot(m1, r - e0), s2 = dot(m2, r - ec);
                if (s0 < -t0 || s1 < -t1 || s2 < -t2) continue;
                if (s0 >= 0.0f && s1 >= 0.0f && s2 >= 0.0f) d = fabsf(dot(n, r));
                else { int rg; f3 q; d = tri_closest<float>(r, e0, ec, n, rg, q); }   // eps margin: exact clamped distance
            }
            if (d < reach) { accepted++; put_min(g, table, scratch, i, j, k, d, G.id); }
        }
    } else if (G.type == 1) {
        // ---- edge wedge: beyond both faces' side planes, between the end caps
        f3 a = ld3(G.f), ab = ld3(G.f + 3) - a, n1 = ld3(G.f + 6), n2 = ld3(G.f + 9);
        float L = sqrtf(dot(ab, ab));
        f3 u = (1.0f / L) * ab;
        f3 w1 = cross(u, n1), w2 = cross(n2, u);
        f3 r0 = mk<float>(x0 - a.x, y - a.y, z - a.z);
        float tu = dot(u, r0), gu = h * u.x;
        clip_ge(tu, gu, -2.0f * eps, tlo, thi);
        clip_ge(-tu, -gu, -(L + 2.0f * eps), tlo, thi);
        clip_ge(dot(w1, r0), h * w1.x, -2.0f * eps, tlo, thi);
        clip_ge(dot(w2, r0), h * w2.x, -2.0f * eps, tlo, thi);
        if (!(tlo <= thi)) return;
        int ia = H.i0 + (int)ceilf(tlo), ib = H.i0 + (int)floorf(thi);
        for (int i = ia; i <= ib; i++) {
            f3 r = mk<float>(fmaf((float)i, h, g.ox) - a.x, r0.y, r0.z);
            tested++;
            float t = dot(u, r);
            if (t < -eps || t > L + eps || dot(w1, r) < -eps || dot(w2, r) < -eps) continue;
            float tc = fminf(fmaxf(t, 0.0f), L);
            f3 q = r - tc * u;
            float d = sqrtf(dot(q, q));
            if (d < reach) { accepted++; put_min(g, table, scratch, i, j, k, d, G.id); }
        }
    } else {
        // ---- vertex cone / hemisphere (eq.10, 362-364)
        f3 v = ld3(G.f), A = ld3(G.f + 3);
        float c = G.f[6];
        float ry = y - v.y, rz = z - v.z;
        float rem = reach * reach - ry * ry - rz * rz;
        if (rem < 0.0f) return;
        float xr = sqrtf(rem), inv_h = 1.0f / h;
        tlo = fmaxf(tlo, (v.x - xr - x0) * inv_h - 1e-2f);
        thi = fminf(thi, (v.x + xr - x0) * inv_h + 1e-2f);
        if (!(tlo <= thi)) return;
        int ia = H.i0 + (int)ceilf(tlo), ib = H.i0 + (int)floorf(thi);
        for (int i = ia; i <= ib; i++) {
            f3 r = mk<float>(fmaf((float)i, h, g.ox) - v.x, ry, rz);
            tested++;
            float d = sqrtf(dot(r, r));
            if (d >= reach || dot(A, r) < c * d - eps) continue;
            accepted++;
            put_min(g, table, scratch, i, j, k, d, G.id);
        }
    }
}

__global__ void __launch_bounds__(EV_BT) evaluate_kernel(MeshView mv, GridParams g, const PolyHdr *__restrict__ hdr,
                                                         const u64 *__restrict__ off, u64 total,
                                                         const int *__restrict__ table, u64 *__restrict__ scratch,
                                                         u64 *__restrict__ ctr) {
    __shared__ u64 s_off[EV_CH + 1];
    __shared__ PolyHdr s_hdr[EV_CH];
    __shared__ Geo s_geo[EV_CH];
    __shared__ int64_t s_plo, s_phi;
    __shared__ u32 s_stat[2];
    const u64 w0 = (u64)blockIdx.x * EV_IPB;
    const u64 w1 = (w0 + EV_IPB < total) ? w0 + EV_IPB : total;
    if (threadIdx.x < 2) {
        // polyhedron holding item w: largest p with off[p] <= w (off is non-decreasing, off[P] = total)
        u64 w = threadIdx.x == 0 ? w0 : w1 - 1;
        int64_t lo = 0, hi = mv.P;          // invariant: off[lo] <= w < off[hi]
        while (hi - lo > 1) {
            int64_t mid = (lo + hi) >> 1;
            if (off[mid] <= w) lo = mid; else hi = mid;
        }
        if (threadIdx.x == 0) { s_plo = lo; s_stat[0] = s_stat[1] = 0; } else s_phi = lo;
    }
    __syncthreads();
    const int64_t plo = s_plo, phi = s_phi;
    u32 tested = 0, accepted = 0;
    for (int64_t q0 = plo; q0 <= phi; q0 += EV_CH) {
        const int cn = (int)((phi - q0 + 1 < EV_CH) ? (phi - q0 + 1) : EV_CH);
        __syncthreads();
        for (int i = threadIdx.x; i <= cn; i += EV_BT) s_off[i] = off[q0 + i];
        for (int i = threadIdx.x; i < cn; i += EV_BT) {
            int64_t p = q0 + i;
            PolyHdr H = hdr[p];
            s_hdr[i] = H;
            if (H.rows) {
                Geo G;
                if (p < mv.F) {
                    const float *T = mv.soup + 9 * p, *N = mv.fn + 3 * p;
#pragma unroll
                    for (int c = 0; c < 9; c++) G.f[c] = T[c];
                    G.f[9] = N[0]; G.f[10] = N[1]; G.f[11] = N[2];
                    G.id = (int)p; G.type = 0;
                } else if (p < (int64_t)mv.F + mv.E) {
                    const EdgeRec &r = mv.erec[p - mv.F];
#pragma unroll
                    for (int c = 0; c < 3; c++) { G.f[c] = r.a[c]; G.f[3 + c] = r.b[c]; G.f[6 + c] = r.n1[c]; G.f[9 + c] = r.n2[c]; }
                    G.id = r.tri; G.type = 1;
                } else {
                    int64_t q = p - mv.F - mv.E;
                    const VertexRec &r = mv.vrec[q >> 1];
                    float sg = (q & 1) ? -1.0f : 1.0f;
#pragma unroll
                    for (int c = 0; c < 3; c++) { G.f[c] = r.pos[c]; G.f[3 + c] = sg * r.axis[c]; }
                    G.f[6] = r.cos_cone;
                    G.id = mv.vmint[q >> 1]; G.type = 2;
                }
                G.pad0 = G.pad1 = 0;
                s_geo[i] = G;
            }
        }
        __syncthreads();
        const u64 lo = s_off[0] > w0 ? s_off[0] : w0;
        const u64 hi = s_off[cn] < w1 ? s_off[cn] : w1;
        for (u64 w = lo + threadIdx.x; w < hi; w += EV_BT) {
            int a = 0, b = cn;              // invariant: s_off[a] <= w < s_off[b]
            while (b - a > 1) {
                int mid = (a + b) >> 1;
                if (s_off[mid] <= w) a = mid; else b = mid;
            }
            process_row(g, s_geo[a], s_hdr[a], (u32)(w - s_off[a]), table, scratch, tested, accepted);
        }
    }
    atomicAdd(&s_stat[0], tested);
    atomicAdd(&s_stat[1], accepted);
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_stat[0]) atomicAdd(&ctr[CTR_TESTED], (u64)s_stat[0]);
        if (s_stat[1]) atomicAdd(&ctr[CTR_ACCEPTED], (u64)s_stat[1]);
    }
}

// ---------------------------------------------------------------------------------------
// A8: sign + emit.  Two kernels: (1) fill_kernel streams the sentinels (+inf, -1;
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

struct CellOut { float d; int t; };

// Populated cell: band decision (fp64 re-check near the band edge) and the sign from the
// pseudonormal of the closest feature of the winning triangle.
__device__ __forceinline__ CellOut finish_cell(const MeshView &mv, const GridParams &g, int i, int j, int k, u64 pack,
                                               u32 &recheck) {
    CellOut o;
    o.d = INFINITY; o.t = -1;
    float d = __uint_as_float((u32)(pack >> 32));
    int t = (int)(u32)pack;
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
    if (fabsf(s) <= 1e-3f * sqrtf(dot(pn, pn) * dot(dv, dv))) redo = true;
    if (redo) {
        // fp64 on the same winning triangle: exact cell position, distance, region, sign
        recheck++;
        V3<double> A = ld3d(T), E0 = ld3d(T + 3) - A, EC = ld3d(T + 6) - A;
        V3<double> Nn = cross(E0, EC);
        Nn = (1.0 / sqrt(dot(Nn, Nn))) * Nn;
        V3<double> X = mk<double>(g.dox + i * g.dh, g.doy + j * g.dh, g.doz + k * g.dh);
        V3<double> Q;
        double D = tri_closest<double>(X - A, E0, EC, Nn, rg, Q);
        if (!(D < g.dband)) return o;                         // strictly inside the band
        V3<double> PN;
        if (rg == RG_FACE) PN = Nn;
        else if (rg <= RG_E2) PN = ld3d(N) + ld3d(mv.fn + 3 * (size_t)(mv.adj[3 * (size_t)t + (rg - RG_E0)] / 3));
        else PN = ld3d(mv.vrec[mv.cvid[3 * (size_t)t + (rg - RG_V0)]].axis);
        neg = dot(PN, (X - A) - Q) < 0.0;
        d = (float)D;
    }
    o.d = (neg && d != 0.0f) ? -d : d;
    o.t = t;
    return o;
}

// One block per active brick (8x8x8 cells, 4 KiB of packed scratch).  Phase 1 loads the
// brick and compacts its populated cells into a shared list; phase 2 spreads the list over
// the threads (the sign pass is the expensive, divergent part); phase 3 writes the brick's
// 64 row segments (8 cells = one 32-B sector each) into both grids.
#define EB_BT 128
__global__ void __launch_bounds__(EB_BT) emit_bricks_kernel(MeshView mv, GridParams g, const int *__restrict__ list,
                                                            const u64 *__restrict__ scratch,
                                                            float *__restrict__ dist, int *__restrict__ tri,
                                                            u64 *__restrict__ ctr) {
    __shared__ __align__(16) u64 s_pack[BRICK_CELLS];
    __shared__ __align__(16) float s_d[BRICK_CELLS];
    __shared__ __align__(16) int s_t[BRICK_CELLS];
    __shared__ unsigned short s_list[BRICK_CELLS];
    __shared__ u32 s_n, s_stat[2];
    const int tid = threadIdx.x;
    if (tid == 0) { s_n = 0; s_stat[0] = s_stat[1] = 0; }
    __syncthreads();
    const int slot = blockIdx.x;
    const int b = list[slot];
    const int bx = b % g.nbx, by = (b / g.nbx) % g.nby, bz = b / (g.nbx * g.nby);
    {
        const ulonglong2 *src = (const ulonglong2 *)(scratch + (size_t)slot * BRICK_CELLS) + 2 * tid;
        ulonglong2 p01 = src[0], p23 = src[1];
        const u64 p[4] = {p01.x, p01.y, p23.x, p23.y};
        const int c0 = 4 * tid;
        // warp-aggregated append of the populated cells
        int cnt = (p[0] != PACK_EMPTY) + (p[1] != PACK_EMPTY) + (p[2] != PACK_EMPTY) + (p[3] != PACK_EMPTY);
        const int lane = tid & 31;
        int inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int v = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += v;
        }
        int base = 0;
        if (lane == 31 && inc) base = (int)atomicAdd(&s_n, (u32)inc);
        base = __shfl_sync(0xffffffffu, base, 31) + inc - cnt;
#pragma unroll
        for (int c = 0; c < 4; c++) {
            s_d[c0 + c] = INFINITY; s_t[c0 + c] = -1;
            if (p[c] != PACK_EMPTY) { s_pack[c0 + c] = p[c]; s_list[base++] = (unsigned short)(c0 + c); }
        }
    }
    __syncthreads();
    const int n = (int)s_n;
    u32 band = 0, recheck = 0;
    for (int q = tid; q < n; q += EB_BT) {
        const int c = s_list[q];
        const int i = bx * 8 + (c & 7), j = by * 8 + ((c >> 3) & 7), k = bz * 8 + (c >> 6);
        CellOut o = finish_cell(mv, g, i, j, k, s_pack[c], recheck);
        s_d[c] = o.d; s_t[c] = o.t;
        band += o.t >= 0;
    }
    __syncthreads();
    {
        const int c0 = 4 * tid;
        const int i = bx * 8 + (c0 & 7), j = by * 8 + ((c0 >> 3) & 7), k = bz * 8 + (c0 >> 6);
        if (j < g.ny && k < g.nz) {
            const size_t o = ((size_t)k * g.ny + j) * g.nx + i;
            if (g.vec4 && i + 3 < g.nx) {
                *(float4 *)(dist + o) = *(const float4 *)(s_d + c0);
                *(int4 *)(tri + o) = *(const int4 *)(s_t + c0);
            } else {
#pragma unroll
                for (int c = 0; c < 4; c++)
                    if (i + c < g.nx) { dist[o + c] = s_d[c0 + c]; tri[o + c] = s_t[c0 + c]; }
            }
        }
    }
    if (band) atomicAdd(&s_stat[0], band);
    if (recheck) atomicAdd(&s_stat[1], recheck);
    __syncthreads();
    if (tid == 0) {
        if (s_stat[0]) atomicAdd(&ctr[CTR_BAND], (u64)s_stat[0]);
        if (s_stat[1]) atomicAdd(&ctr[CTR_RECHECK], (u64)s_stat[1]);
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

int run_compute(sdf_mesh *m, const GridParams &g, float *dist, int *tri, cudaStream_t st) {
    MeshView mv;
    mv.soup = m->soup; mv.fn = m->fn; mv.erec = m->erec; mv.vrec = m->vrec; mv.vmint = m->vmint;
    mv.cvid = m->cvid; mv.adj = m->adj;
    mv.F = (int)m->F; mv.E = (int)m->E; mv.V = (int)m->V;
    mv.P = m->F + m->E + 2 * m->V;
    const int64_t P = mv.P;
    const int64_t nbricks = (int64_t)g.nbx * g.nby * g.nbz;
    int64_t scan_n = P > nbricks ? P : nbricks;
    CKS(ensure(m, &m->hdr, &m->hdr_cap, (size_t)P, st));
    CKS(ensure(m, &m->offsets, &m->offsets_cap, (size_t)P + 1, st));
    CKS(ensure(m, &m->scan_ws, &m->scan_ws_cap, scan_ws_elems(scan_n), st));
    CKS(ensure(m, &m->brick_flag, &m->brick_flag_cap, (size_t)nbricks, st));
    CKS(ensure(m, &m->brick_table, &m->brick_table_cap, (size_t)nbricks, st));
    CKS(ensure(m, &m->brick_list, &m->brick_list_cap, (size_t)nbricks, st));

    // A8a: the sentinel fill depends on nothing: fork it onto the side stream so that it
    // streams to HBM underneath A5-A7 (which are latency / atomic bound)
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    for (int i = SDF_T_CLIP_SCAN; i < SDF_T_COUNT; i++) m->ev_set[i] = false;
    {
        if (!m->side) CK(cudaStreamCreateWithFlags(&m->side, cudaStreamNonBlocking));
        if (!m->ev_fork) CK(cudaEventCreateWithFlags(&m->ev_fork, cudaEventDisableTiming));
        if (!m->ev_join) CK(cudaEventCreateWithFlags(&m->ev_join, cudaEventDisableTiming));
        CK(cudaEventRecord(m->ev_fork, st));
        CK(cudaStreamWaitEvent(m->side, m->ev_fork, 0));
        const int64_t N = (int64_t)g.nx * g.ny * g.nz;
        int64_t fb = (N / 4 + (int64_t)FILL_BT * FILL_UNROLL - 1) / ((int64_t)FILL_BT * FILL_UNROLL);
        if (fb > (int64_t)sms * 2) fb = (int64_t)sms * 2;
        if (fb < 1) fb = 1;
        const int vec = (((uintptr_t)dist & 15) == 0) && (((uintptr_t)tri & 15) == 0);
        stage_mark(m, SDF_T_FILL, 0, m->side);
        KL; fill_kernel<<<(unsigned)fb, FILL_BT, 0, m->side>>>(dist, tri, N, vec);
        stage_mark(m, SDF_T_FILL, 1, m->side);
        CK(cudaEventRecord(m->ev_join, m->side));
    }
    CK(cudaMemsetAsync(m->brick_flag, 0, (size_t)nbricks, st));
    CK(cudaMemsetAsync(m->d_ctr + CTR_POLY, 0, sizeof(u64) * (CTR_COUNT - CTR_POLY), st));

    // A5 + A6: clip, count rows, mark bricks; prefix sums
    stage_mark(m, SDF_T_CLIP_SCAN, 0, st);
    KL; clip_count_kernel<<<(unsigned)((P + 255) / 256), 256, 0, st>>>(mv, g, m->hdr, m->brick_flag);
    KL; count_nonempty_kernel<<<(unsigned)((P + 255) / 256), 256, 0, st>>>(m->hdr, P, m->d_ctr);
    CKS(launch_scan(RowsIn{m->hdr}, RowsOut{m->offsets}, P, m->scan_ws, m->d_ctr + CTR_ITEMS, st));
    KL; set_last_offset_kernel<<<1, 1, 0, st>>>(m->offsets, P, m->d_ctr + CTR_ITEMS);
    CKS(launch_scan(BrickIn{m->brick_flag}, BrickOut{m->brick_table, m->brick_list}, nbricks, m->scan_ws, m->d_ctr + CTR_BRICKS, st));
    CK(cudaGetLastError());

    // host crossing: totals size the launch and the scratch
    u64 tot[2];
    CK(cudaMemcpyAsync(tot, m->d_ctr + CTR_ITEMS, sizeof(tot), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    const u64 items = tot[0], bricks = tot[1];
    stage_mark(m, SDF_T_CLIP_SCAN, 1, st);
    CKS(ensure(m, &m->scratch, &m->scratch_cap, (size_t)(bricks ? bricks : 1) * BRICK_CELLS, st));
    stage_mark(m, SDF_T_CLEAR, 0, st);
    if (bricks) CK(cudaMemsetAsync(m->scratch, 0xFF, (size_t)bricks * BRICK_CELLS * sizeof(u64), st));
    stage_mark(m, SDF_T_CLEAR, 1, st);

    // A7
    if (items) {
        u64 nblk = (items + EV_IPB - 1) / EV_IPB;
        if (nblk > 0x7FFFFFFFull) return SDF_EINVAL;
        stage_mark(m, SDF_T_EVALUATE, 0, st);
        KL; evaluate_kernel<<<(unsigned)nblk, EV_BT, 0, st>>>(mv, g, m->hdr, m->offsets, items, m->brick_table, m->scratch,
                                                         m->d_ctr);
        stage_mark(m, SDF_T_EVALUATE, 1, st);
    }
    // A8b: join the fill, then overwrite the active bricks
    CK(cudaStreamWaitEvent(st, m->ev_join, 0));
    if (bricks) {
        stage_mark(m, SDF_T_EMIT, 0, st);
        KL; emit_bricks_kernel<<<(unsigned)bricks, EB_BT, 0, st>>>(mv, g, m->brick_list, m->scratch, dist, tri, m->d_ctr);
        stage_mark(m, SDF_T_EMIT, 1, st);
    }
    CK(cudaGetLastError());
    m->last_stream = st;
    m->h_ctr[CTR_ITEMS] = items;
    m->h_ctr[CTR_BRICKS] = bricks;
    m->last_bricks_total = nbricks;
    return SDF_OK;
}
