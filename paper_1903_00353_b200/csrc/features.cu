// features.cu -- feature builder (sdf_create): organise the unordered STL-style soup
// (sec.7) into welded vertices, paired half-edges, angle-weighted
// pseudonormals (eq.8) and convex/concave/flat/saddle classes
// (PAPER.md:105-123, 352, 360), and emit the band-independent geometry of the edge wedges
// and vertex cones.
//
// Differences from the paper's design: hashed exact-bit vertex keys instead of
// lossy 30-bit Morton codes, exact (min,max) vertex-id edge keys instead
// of concatenated Morton codes, own radix sort instead of thrust
// (PAPER.md:336), order-independent fixed-point atomics instead of the per-group serial
// regrouping.
#include "primitives.cuh"
#include <math.h>

#define FB 256   // threads per block of the element-wise kernels

static inline unsigned blocks_for(int64_t n, int bt = FB) { return (unsigned)((n + bt - 1) / bt); }

// ---------------------------------------------------------------------------------------
// A0 ingest + A1 weld keys
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ u32 mix32(u32 x, u32 y, u32 z) {
    // 96 -> 32 bit avalanche hash of the exact coordinate bits.  Only has to make equal
    // vertices adjacent after sorting ("the actual order does not matter");
    // equality itself is decided on the exact bits.
    u32 h = x * 0x9E3779B1u;
    h ^= h >> 15; h *= 0x85EBCA77u;
    h ^= y; h *= 0xC2B2AE3Du;
    h ^= h >> 13; h ^= z * 0x27D4EB2Fu;
    h *= 0x165667B1u; h ^= h >> 16; h *= 0x9E3779B1u; h ^= h >> 15;
    return h;
}

// one thread per corner (3 floats): reject non-finite input, canonicalise -0 -> +0, hash
__global__ void __launch_bounds__(FB) ingest_kernel(const float *__restrict__ in, float *__restrict__ soup,
                                                    int ncorner, u32 *__restrict__ keys, u32 *__restrict__ vals,
                                                    int *__restrict__ flags) {
    int c = blockIdx.x * FB + threadIdx.x;
    if (c >= ncorner) return;
    float x = in[3 * (size_t)c], y = in[3 * (size_t)c + 1], z = in[3 * (size_t)c + 2];
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) atomicOr(flags, ERRB_NONFINITE);
    x += 0.0f; y += 0.0f; z += 0.0f;      // -0 + +0 = +0 (round to nearest)
    soup[3 * (size_t)c] = x; soup[3 * (size_t)c + 1] = y; soup[3 * (size_t)c + 2] = z;
    keys[c] = mix32(__float_as_uint(x), __float_as_uint(y), __float_as_uint(z));
    vals[c] = (u32)c;
}

__device__ __forceinline__ bool same_vertex(const float *__restrict__ soup, u32 c0, u32 c1) {
    const u32 *p = (const u32 *)(soup + 3 * (size_t)c0), *q = (const u32 *)(soup + 3 * (size_t)c1);
    return p[0] == q[0] && p[1] == q[1] && p[2] == q[2];
}

// head[s] = 1 iff sorted corner s starts a new vertex (exact bits differ from s-1).
// A new vertex inside an equal-hash run is a hash collision: counted, fixed by weld_fix.
__global__ void __launch_bounds__(FB) weld_flags_kernel(const float *__restrict__ soup, const u32 *__restrict__ keys,
                                                        const u32 *__restrict__ vals, int n,
                                                        unsigned char *__restrict__ head, u64 *__restrict__ ctr) {
    int s = blockIdx.x * FB + threadIdx.x;
    if (s >= n) return;
    bool h = true;
    if (s > 0) {
        h = !same_vertex(soup, vals[s], vals[s - 1]);
        if (h && keys[s] == keys[s - 1]) atomicAdd(&ctr[CTR_WELD_BAD], 1ull);
    }
    head[s] = h ? 1 : 0;
}

__device__ __forceinline__ bool corner_less(const float *__restrict__ soup, u32 c0, u32 c1) {
    const u32 *p = (const u32 *)(soup + 3 * (size_t)c0), *q = (const u32 *)(soup + 3 * (size_t)c1);
    if (p[0] != q[0]) return p[0] < q[0];
    if (p[1] != q[1]) return p[1] < q[1];
    if (p[2] != q[2]) return p[2] < q[2];
    return c0 < c1;
}

// Only does work when a hash collision put distinct vertices in one equal-key run: the
// thread at the head of such a run orders it by the exact bits (insertion sort, runs are
// a few corners long) and recomputes its head flags.  This is the paper's per-group
// regrouping, needed here only for the ~V^2/2^33 colliding pairs.
__global__ void __launch_bounds__(FB) weld_fix_kernel(const float *__restrict__ soup, const u32 *__restrict__ keys,
                                                      u32 *__restrict__ vals, int n, unsigned char *__restrict__ head,
                                                      const u64 *__restrict__ ctr) {
    if (ctr[CTR_WELD_BAD] == 0) return;
    int s = blockIdx.x * FB + threadIdx.x;
    if (s >= n) return;
    if (s > 0 && keys[s] == keys[s - 1]) return;       // not the head of an equal-hash run
    int e = s + 1;
    bool mixed = false;
    while (e < n && keys[e] == keys[s]) { mixed |= (head[e] != 0); e++; }
    if (!mixed) return;
    for (int i = s + 1; i < e; i++) {
        u32 v = vals[i];
        int j = i - 1;
        while (j >= s && corner_less(soup, v, vals[j])) { vals[j + 1] = vals[j]; j--; }
        vals[j + 1] = v;
    }
    for (int i = s + 1; i < e; i++) head[i] = same_vertex(soup, vals[i], vals[i - 1]) ? 0 : 1;
}

struct HeadIn {
    const unsigned char *head;
    __device__ u64 operator()(int64_t i) const { return head[i]; }
};
struct HeadOut {
    const u32 *vals; int *cvid; int *vcorner;
    __device__ void operator()(int64_t i, u64 ex, u64 v) const {
        int vid = (int)(ex + v) - 1;          // inclusive count of heads - 1
        u32 c = vals[i];
        cvid[c] = vid;
        if (v) vcorner[vid] = (int)c;
    }
};

// ---------------------------------------------------------------------------------------
// A3 triangle geometry: unit normal, corner angles, fixed-point pseudonormal accumulation,
// half-edge keys for A2
// ---------------------------------------------------------------------------------------
#define FIXSCALE 1099511627776.0   /* 2^40 */

__device__ __forceinline__ void dcross(const double *a, const double *b, double *r) {
    r[0] = a[1] * b[2] - a[2] * b[1]; r[1] = a[2] * b[0] - a[0] * b[2]; r[2] = a[0] * b[1] - a[1] * b[0];
}
__device__ __forceinline__ double ddot(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

// unit normal in fp64 from the exact fp32 corners; returns false for zero area
__device__ __forceinline__ bool tri_normal64(const float *__restrict__ T, double *n, double p[3][3]) {
#pragma unroll
    for (int k = 0; k < 3; k++)
#pragma unroll
        for (int i = 0; i < 3; i++) p[k][i] = (double)T[3 * k + i];
    double u[3] = {p[1][0] - p[0][0], p[1][1] - p[0][1], p[1][2] - p[0][2]};
    double w[3] = {p[2][0] - p[0][0], p[2][1] - p[0][1], p[2][2] - p[0][2]};
    dcross(u, w, n);
    double L = sqrt(ddot(n, n));
    if (!(L > 0.0)) return false;
    double inv = 1.0 / L;
    n[0] *= inv; n[1] *= inv; n[2] *= inv;
    return true;
}

__global__ void __launch_bounds__(FB) tri_geom_kernel(const float *__restrict__ soup, const int *__restrict__ cvid,
                                                      int F, float *__restrict__ fn, u64 *__restrict__ vacc,
                                                      u64 *__restrict__ ekeys, u32 *__restrict__ evals,
                                                      int *__restrict__ flags) {
    int t = blockIdx.x * FB + threadIdx.x;
    if (t >= F) return;
    const float *T = soup + 9 * (size_t)t;
    int v[3] = {cvid[3 * (size_t)t], cvid[3 * (size_t)t + 1], cvid[3 * (size_t)t + 2]};
    double n[3], p[3][3];
    bool ok = tri_normal64(T, n, p);
    if (!ok || v[0] == v[1] || v[1] == v[2] || v[2] == v[0]) {   // PAPER.md:137 "we disallow faces of zero area"
        atomicOr(flags, ERRB_DEGENERATE);
        n[0] = n[1] = 0.0; n[2] = 1.0;
    }
    fn[3 * (size_t)t] = (float)n[0]; fn[3 * (size_t)t + 1] = (float)n[1]; fn[3 * (size_t)t + 2] = (float)n[2];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        int k1 = (k + 1) % 3, k2 = (k + 2) % 3;
        double u[3] = {p[k1][0] - p[k][0], p[k1][1] - p[k][1], p[k1][2] - p[k][2]};
        double w[3] = {p[k2][0] - p[k][0], p[k2][1] - p[k][1], p[k2][2] - p[k][2]};
        double x[3];
        dcross(u, w, x);
        double alpha = atan2(sqrt(ddot(x, x)), ddot(u, w));          // corner angle, eq.8 weight
        if (ok) {
            // order-independent accumulation: 2^-40 fixed point, two's complement wrap-around
#pragma unroll
            for (int i = 0; i < 3; i++)
                atomicAdd(&vacc[3 * (size_t)v[k] + i], (u64)(long long)llrint(alpha * n[i] * FIXSCALE));
        }
        // half-edge 3t+k goes corner k -> k+1: key = (min vid, max vid)
        u32 a = (u32)v[k], b = (u32)v[k1];
        u32 lo = a < b ? a : b, hi = a < b ? b : a;
        ekeys[3 * (size_t)t + k] = ((u64)lo << 32) | hi;
        evals[3 * (size_t)t + k] = (u32)(3 * t + k);
    }
}

// ---------------------------------------------------------------------------------------
// A2 edge table + A4 edge classes + wedge geometry: one thread per sorted half-edge
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(FB) edge_pair_kernel(const u64 *__restrict__ keys, const u32 *__restrict__ vals,
                                                       int n, const float *__restrict__ soup,
                                                       const float *__restrict__ fn, const int *__restrict__ cvid,
                                                       int *__restrict__ adj, EdgeRec *__restrict__ erec,
                                                       int *__restrict__ flags, u64 *__restrict__ ctr) {
    __shared__ u32 s_cnt[3];
    if (threadIdx.x < 3) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    int s = blockIdx.x * FB + threadIdx.x;
    if (s < n) {
        u64 k = keys[s];
        bool same_prev = (s > 0) && keys[s - 1] == k;
        bool same_next = (s + 1 < n) && keys[s + 1] == k;
        bool even = (s & 1) == 0;
        // closed manifold <=> every key occurs exactly twice <=> runs are aligned pairs
        bool good = even ? (!same_prev && same_next) : (same_prev && !same_next);
        if (!good) atomicOr(flags, ERRB_NOTCLOSED);
        if (good && even) {
            u32 he0 = vals[s], he1 = vals[s + 1];          // he0 < he1 (stable sort)
            // opposite directions <=> the two half-edges start at different vertices
            if (cvid[he0] == cvid[he1]) atomicOr(flags, ERRB_ORIENT);
            adj[he0] = (int)he1;
            adj[he1] = (int)he0;
            int t0 = he0 / 3, k0 = he0 % 3, t1 = he1 / 3;
            const float *A = soup + 9 * (size_t)t0 + 3 * k0, *B = soup + 9 * (size_t)t0 + 3 * ((k0 + 1) % 3);
            {
                // canonical direction a -> b = ascending exact position bits, so the record (and
                // the fp32 rounding of every distance evaluated from it) does not depend on the
                // order of the triangles in the soup; n1 stays the normal of the triangle that
                // traverses a -> b
                const u32 *pa = (const u32 *)A, *pb = (const u32 *)B;
                bool swap = pa[0] != pb[0] ? pa[0] > pb[0] : (pa[1] != pb[1] ? pa[1] > pb[1] : pa[2] > pb[2]);
                if (swap) {
                    int k1 = he1 % 3;
                    t0 = t1; t1 = he0 / 3; k0 = k1;
                    A = soup + 9 * (size_t)t0 + 3 * k0; B = soup + 9 * (size_t)t0 + 3 * ((k0 + 1) % 3);
                }
            }
            const float *N1 = fn + 3 * (size_t)t0, *N2 = fn + 3 * (size_t)t1;
            EdgeRec r;
            double u[3], n1[3], n2[3], x[3];
#pragma unroll
            for (int i = 0; i < 3; i++) {
                r.a[i] = A[i]; r.b[i] = B[i]; r.n1[i] = N1[i]; r.n2[i] = N2[i];
                u[i] = (double)B[i] - (double)A[i]; n1[i] = N1[i]; n2[i] = N2[i];
            }
            double L = sqrt(ddot(u, u));
            dcross(u, n1, x);
            double d = (L > 0.0) ? ddot(x, n2) / L : 0.0;       // PAPER.md:352 d = (ab x n1).n2, normalised
            // flat: the wedge is thinner than 1e-6 * band and lies inside the eps-inflated
            // neighbours (reading #5)
            int cls = d > 1e-6 ? 1 : (d < -1e-6 ? -1 : 0);
            r.tri = t0 < t1 ? t0 : t1;
            r.cls = cls;
            r.pad[0] = r.pad[1] = 0;
            erec[s >> 1] = r;
            atomicAdd(&s_cnt[cls > 0 ? 0 : (cls < 0 ? 1 : 2)], 1u);
        }
    }
    __syncthreads();
    if (threadIdx.x < 3 && s_cnt[threadIdx.x]) atomicAdd(&ctr[CTR_E_CONVEX + threadIdx.x], (u64)s_cnt[threadIdx.x]);
}

// ---------------------------------------------------------------------------------------
// A3/A4 vertices: pseudonormal, cone angle, class
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(FB) vertex_normal_kernel(const u64 *__restrict__ vacc, int V,
                                                           double *__restrict__ vn64) {
    int v = blockIdx.x * FB + threadIdx.x;
    if (v >= V) return;
    double N[3];
#pragma unroll
    for (int i = 0; i < 3; i++) N[i] = (double)(long long)vacc[3 * (size_t)v + i] * (1.0 / FIXSCALE);
    double L = sqrt(ddot(N, N));
    if (L > 1e-9) { N[0] /= L; N[1] /= L; N[2] /= L; }
    else { N[0] = 0.0; N[1] = 0.0; N[2] = 0.0; }      // no usable axis: full sphere on both sides
    vn64[3 * (size_t)v] = N[0]; vn64[3 * (size_t)v + 1] = N[1]; vn64[3 * (size_t)v + 2] = N[2];
}

#define COSSCALE 4503599627370496.0   /* 2^52 */

// one thread per triangle: for each corner, cos of the angle between the face normal and the
// vertex axis (eq.9), which side of the pseudonormal plane the two
// neighbours lie on, lowest incident triangle id
__global__ void __launch_bounds__(FB) vertex_cone_kernel(const float *__restrict__ soup, const int *__restrict__ cvid,
                                                         int F, const double *__restrict__ vn64,
                                                         long long *__restrict__ vcosq, int *__restrict__ vside,
                                                         int *__restrict__ vmint) {
    int t = blockIdx.x * FB + threadIdx.x;
    if (t >= F) return;
    double n[3], p[3][3];
    if (!tri_normal64(soup + 9 * (size_t)t, n, p)) return;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        int v = cvid[3 * (size_t)t + k];
        const double *N = vn64 + 3 * (size_t)v;
        double c = ddot(n, N);
        atomicMin(&vcosq[v], (long long)floor(c * COSSCALE));
        int bits = 0;
#pragma unroll
        for (int q = 1; q <= 2; q++) {
            int kq = (k + q) % 3;
            double e[3] = {p[kq][0] - p[k][0], p[kq][1] - p[k][1], p[kq][2] - p[k][2]};
            double s = ddot(e, N) / sqrt(ddot(e, e));
            bits |= (s > 1e-9) ? 1 : ((s < -1e-9) ? 2 : 4);     // above / below / on the plane
        }
        if ((vside[v] & bits) != bits) atomicOr(&vside[v], bits);
        if (vmint[v] > t) atomicMin(&vmint[v], t);
    }
}

__global__ void __launch_bounds__(FB) vertex_record_kernel(const float *__restrict__ soup,
                                                           const int *__restrict__ vcorner,
                                                           const double *__restrict__ vn64,
                                                           const long long *__restrict__ vcosq,
                                                           const int *__restrict__ vside, int V,
                                                           VertexRec *__restrict__ vrec, u64 *__restrict__ ctr) {
    __shared__ u32 s_cnt[5];
    if (threadIdx.x < 5) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    int v = blockIdx.x * FB + threadIdx.x;
    if (v < V) {
        const float *P = soup + 3 * (size_t)vcorner[v];
        const double *N = vn64 + 3 * (size_t)v;
        double c = (double)vcosq[v] * (1.0 / COSSCALE);
        int side = vside[v];
        bool noaxis = (N[0] == 0.0 && N[1] == 0.0 && N[2] == 0.0);
        int info;
        // convex <=> every neighbour strictly below the pseudonormal plane: only exterior
        // points can be closest to the vertex; concave <=> all strictly above; everything
        // else (saddle, flat, undecided) gets both sides (#2)
        if (side == 2 && !noaxis) info = 1;
        else if (side == 1 && !noaxis) info = 2;
        else info = 3;
        bool hemi = !(c > 0.0) || noaxis;     // ruff: normals span a half space or more
        float cf;
        if (noaxis) cf = -1.0f;               // whole sphere
        else if (hemi) cf = 0.0f;             // hemisphere about the pseudonormal
        else {
            cf = (float)c;
            if ((double)cf > c) cf = nextafterf(cf, -2.0f);
            cf -= 2e-7f;                      // fp32 evaluation slack, widens the cone
        }
        if (hemi) info |= 4;
        // a cone thinner than 1e-6 rad is covered by the eps-inflated neighbours
        bool skip = !hemi && (1.0 - c) < 5e-13;
        if (skip) info = 0;
        VertexRec r;
#pragma unroll
        for (int i = 0; i < 3; i++) { r.pos[i] = P[i]; r.axis[i] = (float)N[i]; }
        r.cos_cone = cf;
        r.info = info;
        vrec[v] = r;
        int slot = skip ? 3 : ((info & 3) == 1 ? 0 : ((info & 3) == 2 ? 1 : 2));
        atomicAdd(&s_cnt[slot], 1u);
        if (hemi && !skip) atomicAdd(&s_cnt[4], 1u);
    }
    __syncthreads();
    if (threadIdx.x < 5 && s_cnt[threadIdx.x]) atomicAdd(&ctr[CTR_V_POS + threadIdx.x], (u64)s_cnt[threadIdx.x]);
}

__global__ void fill_i32_kernel(int *p, int64_t n, int v) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}
__global__ void fill_i64_kernel(long long *p, int64_t n, long long v) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

// ---------------------------------------------------------------------------------------
// host driver
// ---------------------------------------------------------------------------------------
struct TmpPool {     // temporaries of sdf_create, released together
    const sdf_allocator *a; cudaStream_t st; void *p[24]; int n;
    TmpPool(const sdf_allocator *a_, cudaStream_t s) : a(a_), st(s), n(0) {}
    int get(void **out, size_t bytes) {
        int s = dev_alloc(a, out, bytes, st);
        if (s == SDF_OK) p[n++] = *out;
        return s;
    }
    ~TmpPool() { for (int i = n - 1; i >= 0; i--) dev_free(a, p[i], st); }
};

static int status_from_flags(int f) {
    if (f & ERRB_NONFINITE) return SDF_EINVAL;
    if (f & ERRB_DEGENERATE) return SDF_EDEGENERATE;
    if (f & ERRB_NOTCLOSED) return SDF_ENOTCLOSED;
    if (f & ERRB_ORIENT) return SDF_EORIENT;
    return SDF_OK;
}

int build_features(sdf_mesh *m, const float *tri, int on_device, cudaStream_t st) {
    const int64_t F = m->F;
    const int nc = (int)(3 * F);
    const sdf_allocator *al = &m->alloc;
    TmpPool tmp(al, st);

    CKS(dev_alloc(al, (void **)&m->soup, sizeof(float) * 9 * F, st));
    CKS(dev_alloc(al, (void **)&m->fn, sizeof(float) * 3 * F, st));
    CKS(dev_alloc(al, (void **)&m->cvid, sizeof(int) * 3 * F, st));
    CKS(dev_alloc(al, (void **)&m->adj, sizeof(int) * 3 * F, st));
    CKS(dev_alloc(al, (void **)&m->d_ctr, sizeof(u64) * CTR_TOTAL, st));
    CKS(dev_alloc(al, (void **)&m->d_flags, sizeof(int) * 4, st));
    CK(cudaMemsetAsync(m->d_ctr, 0, sizeof(u64) * CTR_TOTAL, st));
    CK(cudaMemsetAsync(m->d_flags, 0, sizeof(int) * 4, st));
    CK(cudaMemsetAsync(m->adj, 0xFF, sizeof(int) * 3 * F, st));

    // ---- A0: ingest
    stage_mark(m, SDF_T_INGEST_WELD, 0, st);
    const float *src = tri;
    float *staging = nullptr;
    if (!on_device) {
        CKS(tmp.get((void **)&staging, sizeof(float) * 9 * F));
        CK(cudaMemcpyAsync(staging, tri, sizeof(float) * 9 * F, cudaMemcpyHostToDevice, st));
        src = staging;
    }
    u32 *k32a, *k32b, *va, *vb, *hist;
    u64 *scan_ws;
    unsigned char *head;
    int *vcorner;
    CKS(tmp.get((void **)&k32a, sizeof(u32) * nc));
    CKS(tmp.get((void **)&k32b, sizeof(u32) * nc));
    CKS(tmp.get((void **)&va, sizeof(u32) * nc));
    CKS(tmp.get((void **)&vb, sizeof(u32) * nc));
    CKS(tmp.get((void **)&hist, sizeof(u32) * radix_hist_elems(nc)));
    size_t ws_elems = scan_ws_elems((int64_t)nc > (int64_t)radix_hist_elems(nc) ? (int64_t)nc : (int64_t)radix_hist_elems(nc));
    CKS(tmp.get((void **)&scan_ws, sizeof(u64) * ws_elems));
    CKS(tmp.get((void **)&head, (size_t)nc));
    CKS(tmp.get((void **)&vcorner, sizeof(int) * nc));      // V <= 3F
    KL; ingest_kernel<<<blocks_for(nc), FB, 0, st>>>(src, m->soup, nc, k32a, va, m->d_flags);

    // ---- A1: weld (radix sort of the hashed keys, exact compare of neighbours)
    {
        const int shifts[4] = {0, 8, 16, 24};
        bool first;
        CKS(radix_sort_pairs<u32>(k32a, va, k32b, vb, nc, shifts, 4, hist, scan_ws, st, &first));
        u32 *ks = first ? k32a : k32b, *vs = first ? va : vb;
        KL; weld_flags_kernel<<<blocks_for(nc), FB, 0, st>>>(m->soup, ks, vs, nc, head, m->d_ctr);
        KL; weld_fix_kernel<<<blocks_for(nc), FB, 0, st>>>(m->soup, ks, vs, nc, head, m->d_ctr);
        HeadIn hin{head};
        HeadOut hout{vs, m->cvid, vcorner};
        CKS(launch_scan(hin, hout, (int64_t)nc, scan_ws, m->d_ctr + CTR_V, st));
    }
    stage_mark(m, SDF_T_INGEST_WELD, 1, st);
    // first host crossing: the vertex count sizes every per-vertex table
    CK(cudaMemcpyAsync(m->h_ctr, m->d_ctr, sizeof(u64) * CTR_COUNT, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    m->V = (int64_t)m->h_ctr[CTR_V];
    const int V = (int)m->V;

    // ---- A3 (per triangle) + half-edge keys
    stage_mark(m, SDF_T_EDGES, 0, st);
    u64 *vacc, *eka, *ekb;
    CKS(tmp.get((void **)&vacc, sizeof(u64) * 3 * (size_t)V));
    CKS(tmp.get((void **)&eka, sizeof(u64) * nc));
    CKS(tmp.get((void **)&ekb, sizeof(u64) * nc));
    CK(cudaMemsetAsync(vacc, 0, sizeof(u64) * 3 * (size_t)V, st));
    KL; tri_geom_kernel<<<blocks_for(F), FB, 0, st>>>(m->soup, m->cvid, (int)F, m->fn, vacc, eka, va, m->d_flags);

    // ---- A2: edge table (radix sort of the (min,max) keys over their significant bits)
    {
        int bits = 1;
        while (((int64_t)1 << bits) < (int64_t)V) bits++;          // vertex ids < V
        int shifts[8], np = 0;
        for (int b = 0; b < bits; b += 8) shifts[np++] = b;
        for (int b = 0; b < bits; b += 8) shifts[np++] = 32 + b;
        bool first;
        CKS(radix_sort_pairs<u64>(eka, va, ekb, vb, nc, shifts, np, hist, scan_ws, st, &first));
        u64 *ks = first ? eka : ekb;
        u32 *vs = first ? va : vb;
        if (nc & 1) {
            int f = ERRB_NOTCLOSED;
            CK(cudaMemcpyAsync(m->d_flags, &f, sizeof(int), cudaMemcpyHostToDevice, st));
        }
        m->E = nc / 2;
        CKS(dev_alloc(al, (void **)&m->erec, sizeof(EdgeRec) * (size_t)(m->E > 0 ? m->E : 1), st));
        KL; edge_pair_kernel<<<blocks_for(nc), FB, 0, st>>>(ks, vs, nc & ~1, m->soup, m->fn, m->cvid, m->adj, m->erec,
                                                        m->d_flags, m->d_ctr);
    }
    CK(cudaGetLastError());
    stage_mark(m, SDF_T_EDGES, 1, st);

    // ---- A3/A4 vertices (garbage-in on invalid input is harmless: ids stay in range)
    stage_mark(m, SDF_T_VERTICES, 0, st);
    double *vn64;
    long long *vcosq;
    int *vside;
    CKS(tmp.get((void **)&vn64, sizeof(double) * 3 * (size_t)V));
    CKS(tmp.get((void **)&vcosq, sizeof(long long) * (size_t)V));
    CKS(tmp.get((void **)&vside, sizeof(int) * (size_t)V));
    CKS(dev_alloc(al, (void **)&m->vmint, sizeof(int) * (size_t)V, st));
    CKS(dev_alloc(al, (void **)&m->vrec, sizeof(VertexRec) * (size_t)V, st));
    KL; vertex_normal_kernel<<<blocks_for(V), FB, 0, st>>>(vacc, V, vn64);
    KL; fill_i64_kernel<<<blocks_for(V), FB, 0, st>>>(vcosq, V, 0x7FFFFFFFFFFFFFFFll);
    KL; fill_i32_kernel<<<blocks_for(V), FB, 0, st>>>(m->vmint, V, 0x7FFFFFFF);
    CK(cudaMemsetAsync(vside, 0, sizeof(int) * (size_t)V, st));
    KL; vertex_cone_kernel<<<blocks_for(F), FB, 0, st>>>(m->soup, m->cvid, (int)F, vn64, vcosq, vside, m->vmint);
    KL; vertex_record_kernel<<<blocks_for(V), FB, 0, st>>>(m->soup, vcorner, vn64, vcosq, vside, V, m->vrec, m->d_ctr);
    CK(cudaGetLastError());
    stage_mark(m, SDF_T_VERTICES, 1, st);
    // second host crossing: validation flags + class counters
    int hflags[4];
    CK(cudaMemcpyAsync(hflags, m->d_flags, sizeof(hflags), cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(m->h_ctr, m->d_ctr, sizeof(u64) * CTR_COUNT, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));      // temporaries are released after this point
    return status_from_flags(hflags[0]);
}
