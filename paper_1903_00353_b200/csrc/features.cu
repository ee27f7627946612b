// features.cu -- feature builder (sdf_create): organise the unordered STL-style soup
// (sec.7) into welded vertices, paired half-edges, angle-weighted
// pseudonormals (eq.8) and convex/concave/flat/saddle classes
// (PAPER.md:105-123, 352, 360), and emit the band-independent geometry of the edge wedges
// and vertex cones.
//
// Differences from the paper's design: hashed exact-bit vertex keys instead of
// lossy 30-bit Morton codes, exact (min,max) vertex-id edge keys instead
// of concatenated Morton codes, a one-pass counting sort of the triangles by a
// fine Morton bin instead of thrust::sort_by_key on the features, order-independent
// fixed-point atomics instead of the per-group serial regrouping.
#include "primitives.cuh"
#include "evaluate.cuh"
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define FB 256   // threads per block of the element-wise kernels
#ifndef TG_MINB
#define TG_MINB 5 // resident blocks per SM asked of the fp64-heavy per-triangle kernels (latency bound)
#endif

static inline unsigned blocks_for(int64_t n, int bt = FB) { return (unsigned)((n + bt - 1) / bt); }

// ---------------------------------------------------------------------------------------
// A0 ingest + A1 weld: open-addressing hash table keyed by the exact coordinate bits
// ---------------------------------------------------------------------------------------
#define EMPTY32 0xFFFFFFFFu
#define HE_MATCHED 0x80000000u

__device__ __forceinline__ u32 mix32(u32 x, u32 y, u32 z) {
    // 96 -> 32 bit avalanche hash.  It only spreads the keys over the table
    // ("the actual order does not matter"); equality is decided on the exact bits.
    u32 h = x * 0x9E3779B1u;
    h ^= h >> 15; h *= 0x85EBCA77u;
    h ^= y; h *= 0xC2B2AE3Du;
    h ^= h >> 13; h ^= z * 0x27D4EB2Fu;
    h *= 0x165667B1u; h ^= h >> 16; h *= 0x9E3779B1u; h ^= h >> 15;
    return h;
}

// ---- spatial binning (A0).  The soup arrives in arbitrary order; every later
// step gathers and scatters by vertex / edge / cell, so the library works on a copy ordered
// along a coarse Morton curve (the paper sorts by Morton code for the same reason,
// PAPER.md:296-332).  The order is internal: ids written to the output are the caller's.
__device__ __forceinline__ int f2ord(float f) {           // monotone float -> int
    int i = __float_as_int(f);
    return i >= 0 ? i : i ^ 0x7FFFFFFF;
}
__device__ __forceinline__ float ord2f(int i) { return __int_as_float(i >= 0 ? i : i ^ 0x7FFFFFFF); }

// approximate bounding box from a strided sample of first corners (only steers the binning)
__global__ void __launch_bounds__(FB) bbox_sample_kernel(const float *__restrict__ in, int F, int stride,
                                                         int *__restrict__ bbox) {
    int t = (blockIdx.x * FB + threadIdx.x) * stride;
    int lo[3] = {0x7FFFFFFF, 0x7FFFFFFF, 0x7FFFFFFF}, hi[3] = {(int)0x80000000, (int)0x80000000, (int)0x80000000};
    if (t < F) {
        const float *p = in + 9 * (size_t)t;
#pragma unroll
        for (int i = 0; i < 3; i++)
            if (isfinite(p[i])) { lo[i] = hi[i] = f2ord(p[i]); }
    }
#pragma unroll
    for (int i = 0; i < 3; i++) {
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            lo[i] = min(lo[i], __shfl_xor_sync(0xffffffffu, lo[i], o));
            hi[i] = max(hi[i], __shfl_xor_sync(0xffffffffu, hi[i], o));
        }
        if ((threadIdx.x & 31) == 0) { atomicMin(&bbox[i], lo[i]); atomicMax(&bbox[3 + i], hi[i]); }
    }
}

__global__ void __launch_bounds__(FB) identity_perm_kernel(int F, u32 *__restrict__ perm) {
    int t = blockIdx.x * FB + threadIdx.x;
    if (t < F) perm[t] = (u32)t;
}

// ---- tile builder: ONE-pass counting sort by a fine Morton bin (up to 7 bits per axis).  Only a 4-byte index moves
// (the triangles themselves are gathered by tile_weld_kernel), so a bin's slot is handed out by an atomic ticket and
// the bin offsets come from one scan over the bins.  Inside a bin the order is the order of arrival -- it differs from
// run to run and nothing that reaches the output depends on it.
__device__ __forceinline__ u32 spread3_10(u32 v) {         // 10 bits -> every third bit
    v &= 0x3FFu;
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}
// Morton bin of a position: `bits` bits per axis over the sampled box (a function of the position alone)
__device__ __forceinline__ u32 fine_bin_of(float x, float y, float z, const int *__restrict__ bbox, int bits) {
    const float nb = (float)(1 << bits);
    const float p[3] = {x, y, z};
    u32 q[3];
#pragma unroll
    for (int i = 0; i < 3; i++) {
        const float lo = ord2f(bbox[i]), hi = ord2f(bbox[3 + i]);
        const float w = hi - lo;
        float f = (w > 0.0f && isfinite(w)) ? (p[i] - lo) / w * nb : 0.0f;
        f = fminf(fmaxf(f, 0.0f), nb - 1.0f);                 // NaN -> 0; outliers -> end bins
        q[i] = (u32)f;
    }
    return spread3_10(q[0]) | (spread3_10(q[1]) << 1) | (spread3_10(q[2]) << 2);
}
__global__ void __launch_bounds__(FB) fine_bin_kernel(const float *__restrict__ in, int F, const int *__restrict__ bbox,
                                                      int bits, u32 *cnt, u32 *__restrict__ key, u32 *__restrict__ ticket) {
    int t = blockIdx.x * FB + threadIdx.x;
    if (t >= F) return;
    const float *p = in + 9 * (size_t)t;
    const u32 k = fine_bin_of(p[0], p[1], p[2], bbox, bits);
    key[t] = k;
    ticket[t] = atomicAdd(&cnt[k], 1u);
}
struct BinIn {
    const u32 *c;
    __device__ u64 operator()(int64_t i) const { return c[i]; }
};
struct BinOut {
    u32 *c;
    __device__ void operator()(int64_t i, u64 ex, u64) const { c[i] = (u32)ex; }
};
__global__ void __launch_bounds__(FB) fine_scatter_kernel(int F, const u32 *__restrict__ base, const u32 *__restrict__ key,
                                                          const u32 *__restrict__ ticket, u32 *__restrict__ perm) {
    int t = blockIdx.x * FB + threadIdx.x;
    if (t < F) perm[base[key[t]] + ticket[t]] = (u32)t;
}

__device__ __forceinline__ u32 canon_bits(float x) { return __float_as_uint(x + 0.0f); }   // -0 + +0 = +0

// The global weld table, laid out along the sorted order of the triangles: the home slot of a position is the start of
// its Morton bin in that order (the exclusive bin counts of the counting sort) scaled to the table, plus a hash over the bin's share of the table.
// The corners of a bin, welded at about the same time, then probe one small region of the table (L2 hits instead of
// DRAM round trips); after WTAB_LOCAL probes without success the sequence continues at the uniformly hashed position.
struct WeldTab { u32 *tab; u32 mask; u32 scale; const u32 *base; const int *bbox; int bits; u32 nf; };
#define WTAB_LOCAL 64
__device__ __forceinline__ u32 wtab_home(const WeldTab &w, float x, float y, float z, u32 bx, u32 by, u32 bz) {
    const u32 hs = mix32(bx, by, bz);
    if (!w.scale) return hs & w.mask;
    // the bin's region: [base[b], base[b+1]) triangles scaled to the table (~4 slots per triangle, two vertices per
    // four triangles: load 1/8 everywhere, also in the bins at the poles of a UV mesh that hold thousands of vertices)
    const u32 b = fine_bin_of(x, y, z, w.bbox, w.bits);
    const u32 b0 = w.base[b], b1 = (b + 1u < (1u << (3 * w.bits))) ? w.base[b + 1u] : w.nf;
    const u32 lo = (u32)(((u64)b0 * w.scale) >> 12), len = (u32)(((u64)(b1 - b0) * w.scale) >> 12) + 16u;
    return (lo + (u32)(((u64)hs * len) >> 32)) & w.mask;
}
__device__ __forceinline__ void wtab_next(const WeldTab &w, u32 bx, u32 by, u32 bz, u32 &h, int &n) {
    n++;
    if (w.scale && n == WTAB_LOCAL) h = mix32(bx, by, bz) & w.mask;
    else h = (h + 1) & w.mask;
}

// One thread per corner of the internal order: gather the corner from the caller's soup
// (reject non-finite input, canonicalise -0 -> +0, write the internal copy), then find-or-insert
// its vertex in the weld table (linear probing).  A slot holds a corner index of its vertex;
// identity is checked on the exact bits of that corner in the immutable input (its sector was
// just read by the thread that owns it, so the check hits L2).  The corner that inserts a vertex
// takes its id from a counter (one atomicAdd per block), resets the vertex' accumulators and leaves
// the id in wvid[slot]; slot[c] = table position of c, resolved to ids by tri_geom_kernel.  (The ids
// depend on the order in which warps run; nothing that reaches the output does.)
__global__ void __launch_bounds__(FB) ingest_weld_kernel(const float *__restrict__ in, const int *__restrict__ perm,
                                                         int ncorner, float *__restrict__ soup,
                                                         int *__restrict__ inv_perm, WeldTab wt,
                                                         u32 *__restrict__ slot, u32 *__restrict__ wvid,
                                                         int *__restrict__ vcorner, u64 *__restrict__ vacc,
                                                         long long *__restrict__ vcosq, long long *__restrict__ vcospos,
                                                         int *__restrict__ vside, int *__restrict__ vmint, int vcap,
                                                         u64 *ctr, int *__restrict__ flags, int *__restrict__ perm_identity) {
    // perm == nullptr: the internal order is the caller's (small meshes are not sorted) and perm_identity is filled here
    __shared__ u32 s_nins, s_base;
    if (threadIdx.x == 0) s_nins = 0;
    __syncthreads();
    const int c = blockIdx.x * FB + threadIdx.x;
    bool inserted = false;
    u32 h = 0;
    if (c < ncorner) {
        const int i = c / 3, k = c - 3 * i;
        const int t = perm ? perm[i] : i;
        if (!perm && k == 0) perm_identity[i] = i;
        const float *p = in + 9 * (size_t)t + 3 * k;
        float x = p[0], y = p[1], z = p[2];
        if (!(isfinite(x) && isfinite(y) && isfinite(z))) atomicOr(flags, ERRB_NONFINITE);
        x += 0.0f; y += 0.0f; z += 0.0f;
        soup[3 * (size_t)c] = x; soup[3 * (size_t)c + 1] = y; soup[3 * (size_t)c + 2] = z;
        if (k == 0) inv_perm[t] = i;
        const u32 bx = __float_as_uint(x), by = __float_as_uint(y), bz = __float_as_uint(z);
        h = wtab_home(wt, x, y, z, bx, by, bz);
        int np = 0;
        for (;;) {
            u32 cur = __ldcg(wt.tab + h);
            if (cur == EMPTY32) {
                cur = atomicCAS(wt.tab + h, EMPTY32, (u32)c);
                if (cur == EMPTY32) { inserted = true; break; }
            }
            const int ci = (int)cur / 3, ck = (int)cur - 3 * ci;
            const float *q = in + 9 * (size_t)(perm ? perm[ci] : ci) + 3 * ck;
            if (canon_bits(q[0]) == bx && canon_bits(q[1]) == by && canon_bits(q[2]) == bz) break;
            wtab_next(wt, bx, by, bz, h, np);
        }
        slot[c] = h;
    }
    // vertex ids: one atomicAdd on the global counter per BLOCK (one per warp serialises 4e5 same-address atomics at
    // C4: +0.2 ms); ranks inside the block by a shared-memory counter
    const unsigned ins = __ballot_sync(0xffffffffu, inserted);
    const int lane = threadIdx.x & 31;
    u32 wbase = 0;
    if (ins && lane == __ffs(ins) - 1) wbase = atomicAdd(&s_nins, (u32)__popc(ins));
    __syncthreads();
    if (threadIdx.x == 0 && s_nins) s_base = (u32)atomicAdd(&ctr[CTR_V], (u64)s_nins);
    __syncthreads();
    if (ins) wbase = __shfl_sync(0xffffffffu, wbase, __ffs(ins) - 1);
    if (inserted) {
        const u32 vid = s_base + wbase + (u32)__popc(ins & ((1u << lane) - 1u));
        if (vid >= (u32)vcap) {
            // more vertices than a closed surface of F triangles can have (V <= 3F/2): the tables are not that large
            atomicOr(flags, ERRB_NOTCLOSED);
            wvid[h] = (u32)(vcap - 1);
        } else {
            wvid[h] = vid;
            vcorner[vid] = c;
            vacc[3 * (size_t)vid] = 0ull; vacc[3 * (size_t)vid + 1] = 0ull; vacc[3 * (size_t)vid + 2] = 0ull;
            vcosq[vid] = 0x7F7F7F7F7F7F7F7Fll;
            if (vcospos) vcospos[vid] = 0x7F7F7F7F7F7F7F7Fll;
            vside[vid] = 0;
            vmint[vid] = 0x7F7F7F7F;
        }
    }
}

// ---------------------------------------------------------------------------------------
// A3 triangle geometry: corner -> vertex ids, unit normal, corner angles, fixed-point
// pseudonormal accumulation, number of forward half-edges (for the edge ids of A2)
// ---------------------------------------------------------------------------------------
#define FIXSCALE 1099511627776.0   /* 2^40 */
#define COSSCALE 4503599627370496.0   /* 2^52 */

__device__ __forceinline__ u32 edge_hash(u32 u, u32 w) { return mix32(u, w, 0x51ED270Bu); }

__device__ __forceinline__ int he_next(int he) { int k = he % 3; return he - k + (k == 2 ? 0 : k + 1); }

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

#include "tile_features.cuh"

// ===================================================================================================
// the global-table builder (default): every corner / half-edge through hash tables in global memory
// ===================================================================================================
__global__ void __launch_bounds__(FB, TG_MINB) tri_geom_kernel(const float *__restrict__ soup, const u32 *__restrict__ wvid,
                                                      const u32 *__restrict__ slot, int F, int *__restrict__ cvid,
                                                      float *__restrict__ fn, u64 *__restrict__ vacc,
                                                      u32 *etab, u32 emask, int *__restrict__ flags,
                                                      const GridParams *__restrict__ mark_g,
                                                      unsigned char *__restrict__ brick_flag,
                                                      int *__restrict__ adj, float *__restrict__ fsm) {
    int t = blockIdx.x * FB + threadIdx.x;
    if (t >= F) return;
    // what the pairing kernel (next on this stream) expects: no partner yet, no smooth edge absorbed yet
    adj[3 * (size_t)t] = -1; adj[3 * (size_t)t + 1] = -1; adj[3 * (size_t)t + 2] = -1;
    fsm[t] = 0.0f;
    const float *T = soup + 9 * (size_t)t;
    int v[3];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        v[k] = (int)wvid[slot[3 * (size_t)t + k]];
        cvid[3 * (size_t)t + k] = v[k];
    }
    // forward half-edges (ascending ids): the first probe of each is loaded now and waited for after the fp64 work
    u32 eh[3], ecur[3];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const int k1 = (k + 1) % 3;
        eh[k] = edge_hash((u32)v[k], (u32)v[k1]) & emask;
        ecur[k] = (v[k] < v[k1]) ? __ldcg(etab + eh[k]) : 0u;
    }
    double n[3], p[3][3];
    bool ok = tri_normal64(T, n, p);
    // PAPER.md:137 "we disallow faces of zero area".  (A repeated vertex IS a zero area, exactly: equal corners give a zero
    // cross product.  The ids are not consulted: past the capacity of the vertex tables they are clamped.)
    if (!ok) {
        atomicOr(flags, ERRB_DEGENERATE);
        n[0] = n[1] = 0.0; n[2] = 1.0;
    }
    const float nf[3] = {(float)n[0], (float)n[1], (float)n[2]};
    fn[3 * (size_t)t] = nf[0]; fn[3 * (size_t)t + 1] = nf[1]; fn[3 * (size_t)t + 2] = nf[2];
    // sdf_transform (the grid is known already): A6a's brick marks while the corners and the normal are in registers
    if (mark_g) mark_triangle_bricks(*mark_g, T, nf, brick_flag);
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
    }
    // half-edge 3t+k goes corner k -> k+1; forward = ascending ids.  Forward
    // half-edges take the first empty slot of the edge table on their probe sequence (no key
    // check: a valid mesh has one forward half-edge per key, and a duplicate just leaves an
    // entry nobody claims, which the pair count exposes).  The three first claims go out together.
    // (a table laid out along the vertex ids, so that the probes of an edge's two triangles hit L2, was measured:
    // it halves the DRAM reads of the two edge kernels and makes them slower -- their stalls are the round
    // trips of the L2 atomics themselves, and clustered homes lengthen the probe sequences)
    u32 got[3];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const int k1 = (k + 1) % 3;
        got[k] = EMPTY32;                                    // EMPTY32 = placed (or not a forward half-edge)
        if (v[k] < v[k1]) got[k] = (ecur[k] == EMPTY32) ? atomicCAS(etab + eh[k], EMPTY32, (u32)(3 * t + k)) : ecur[k];
    }
#pragma unroll
    for (int k = 0; k < 3; k++) {
        if (got[k] == EMPTY32) continue;
        u32 h = eh[k];
        do h = (h + 1) & emask;
        while (__ldcg(etab + h) != EMPTY32 || atomicCAS(etab + h, EMPTY32, (u32)(3 * t + k)) != EMPTY32);
    }
}

// ---- exact classification of an invalid edge table (error path only): sort the (min,max)
// keys, a closed manifold has every key exactly twice (aligned pairs) in opposite directions
__global__ void __launch_bounds__(FB) edge_keys_kernel(const int *__restrict__ cvid, int n, u64 *__restrict__ keys,
                                                       u32 *__restrict__ vals) {
    int he = blockIdx.x * FB + threadIdx.x;
    if (he >= n) return;
    u32 a = (u32)cvid[he], b = (u32)cvid[he_next(he)];
    u32 lo = a < b ? a : b, hi = a < b ? b : a;
    keys[he] = ((u64)lo << 32) | hi;
    vals[he] = (u32)he;
}
__global__ void __launch_bounds__(FB) edge_validate_kernel(const u64 *__restrict__ keys, const u32 *__restrict__ vals,
                                                           int n, const int *__restrict__ cvid, int *__restrict__ flags) {
    int s = blockIdx.x * FB + threadIdx.x;
    if (s >= n) return;
    u64 k = keys[s];
    bool same_prev = (s > 0) && keys[s - 1] == k;
    bool same_next = (s + 1 < n) && keys[s + 1] == k;
    bool even = (s & 1) == 0;
    bool good = even ? (!same_prev && same_next) : (same_prev && !same_next);
    if (!good) atomicOr(flags, ERRB_NOTCLOSED);
    // opposite directions <=> the two half-edges start at different vertices
    if (good && even && cvid[vals[s]] == cvid[vals[s + 1]]) atomicOr(flags, ERRB_ORIENT);
}

// ---------------------------------------------------------------------------------------
// A3/A4 vertices: pseudonormal, cone angle, class
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(FB) vertex_normal_kernel(const u64 *__restrict__ vacc, int V, const u64 *__restrict__ vcount,
                                                           double *__restrict__ vn64) {
    int v = blockIdx.x * FB + threadIdx.x;
    if (vcount) V = min(V, (int)*vcount);
    if (v >= V) return;
    double N[3];
#pragma unroll
    for (int i = 0; i < 3; i++) N[i] = (double)(long long)vacc[3 * (size_t)v + i] * (1.0 / FIXSCALE);
    double L = sqrt(ddot(N, N));
    if (L > 1e-9) { N[0] /= L; N[1] /= L; N[2] /= L; }
    else { N[0] = 0.0; N[1] = 0.0; N[2] = 0.0; }      // no usable axis: full sphere on both sides
    vn64[3 * (size_t)v] = N[0]; vn64[3 * (size_t)v + 1] = N[1]; vn64[3 * (size_t)v + 2] = N[2];
}

// one thread per triangle: for each corner, cos of the angle between the face normal and the
// vertex axis (eq.9), which side of the pseudonormal plane the two
// neighbours lie on, lowest incident triangle id
__global__ void __launch_bounds__(FB, TG_MINB) vertex_cone_kernel(const float *__restrict__ soup, const int *__restrict__ cvid,
                                                         int F, const double *__restrict__ vn64,
                                                         long long *__restrict__ vcosq, int *__restrict__ vside,
                                                         const int *__restrict__ perm, int *__restrict__ vmint,
                                                         long long *__restrict__ vcospos) {
    int t = blockIdx.x * FB + threadIdx.x;
    if (t >= F) return;
    double n[3], p[3][3];
    if (!tri_normal64(soup + 9 * (size_t)t, n, p)) return;
    const int xt = perm[t];                               // the caller's triangle id
#pragma unroll
    for (int k = 0; k < 3; k++) {
        int v = cvid[3 * (size_t)t + k];
        const double *N = vn64 + 3 * (size_t)v;
        double c = ddot(n, N);
        atomicMin(&vcosq[v], (long long)floor(c * COSSCALE));
        // ablation: the cone over the positive-pointing normals only
        if (vcospos && c > 0.0) atomicMin(&vcospos[v], (long long)floor(c * COSSCALE));
        int bits = 0;
#pragma unroll
        for (int q = 1; q <= 2; q++) {
            int kq = (k + q) % 3;
            double e[3] = {p[kq][0] - p[k][0], p[kq][1] - p[k][1], p[kq][2] - p[k][2]};
            double s = ddot(e, N) / sqrt(ddot(e, e));
            bits |= (s > 1e-9) ? 1 : ((s < -1e-9) ? 2 : 4);     // above / below / on the plane
        }
        if ((vside[v] & bits) != bits) atomicOr(&vside[v], bits);
        if (vmint[v] > xt) atomicMin(&vmint[v], xt);
    }
}

// vn64 == nullptr: the axis is normalised here from the fixed-point sums vacc; vcount != nullptr: the number of
// vertices is read on the device (the tile builder launches for the capacity of the tables)
__global__ void __launch_bounds__(FB) vertex_record_kernel(const float *__restrict__ soup,
                                                           const int *__restrict__ vcorner,
                                                           const double *__restrict__ vn64, const u64 *__restrict__ vacc,
                                                           const u64 *__restrict__ vcount,
                                                           const long long *__restrict__ vcosq,
                                                           const int *__restrict__ vside, int V,
                                                           const long long *__restrict__ vcospos, float smooth_sin,
                                                           VertexRec *__restrict__ vrec, unsigned char *__restrict__ vsm,
                                                           u32 *__restrict__ cone_list, u64 *__restrict__ ctr) {
    __shared__ u32 s_cnt[5], s_live, s_base;
    if (threadIdx.x < 5) s_cnt[threadIdx.x] = 0;
    if (threadIdx.x == 5) s_live = 0;
    __syncthreads();
    int v = blockIdx.x * FB + threadIdx.x;
    int sides = 0, rank = 0;
    if (vcount) V = min(V, (int)*vcount);
    if (v < V) {
        const float *P = soup + 3 * (size_t)vcorner[v];
        double Nl[3];
        const double *N = Nl;
        if (vn64) N = vn64 + 3 * (size_t)v;
        else vertex_axis64(vacc, (size_t)v, Nl);
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
        else if (hemi && vcospos && vcospos[v] != 0x7F7F7F7F7F7F7F7Fll) {
            // ablation: "a cone of positive pointing normals is sufficient in practice"
            const double cp = (double)vcospos[v] * (1.0 / COSSCALE);
            cf = (float)cp;
            if ((double)cf > cp) cf = nextafterf(cf, -2.0f);
            cf -= 2e-7f;
        } else if (hemi) cf = 0.0f;           // hemisphere about the pseudonormal
        else {
            cf = (float)c;
            if ((double)cf > c) cf = nextafterf(cf, -2.0f);
            cf -= 2e-7f;                      // fp32 evaluation slack, widens the cone
        }
        if (hemi) info |= 4;
        // a cone thinner than 1e-6 rad is covered by the eps-inflated neighbours
        bool skip = !hemi && (1.0 - c) < 5e-13;
        // smooth: the whole cone of normals within asin(smooth_sin) / 2 of the axis.  No cone; the incident faces
        // widen their prisms by reach * sin(2 theta) instead (evaluate.cuh face_margin_sin reads it back from cos_cone)
        // (also the cones thinner than 1e-6 rad, skipped above: their margin is the smallest the byte code holds)
        const float s2 = (hemi || noaxis) ? INFINITY : cone_sin2(cf);
        if (s2 <= smooth_sin && s2 * VSM_SCALE <= 255.0f) skip = true;       // (the byte code must hold it, rounded up)
        if (skip) info = 8;
        vsm[v] = skip ? (unsigned char)min(255, max(1, (int)ceilf(s2 * VSM_SCALE))) : (unsigned char)0;
        VertexRec r;
#pragma unroll
        for (int i = 0; i < 3; i++) { r.pos[i] = P[i]; r.axis[i] = (float)N[i]; }
        r.cos_cone = cf;
        r.info = info;
        vrec[v] = r;
        int slot = skip ? 3 : ((info & 3) == 1 ? 0 : ((info & 3) == 2 ? 1 : 2));
        atomicAdd(&s_cnt[slot], 1u);
        if (hemi && !skip) atomicAdd(&s_cnt[4], 1u);
        // the cones that exist: one entry per emitted side (a vertex without axis is one whole ball: + side only)
        sides = skip ? 0 : (cf <= -1.0f ? 1 : (info & 3));
        if (sides) rank = (int)atomicAdd(&s_live, (u32)__popc(sides));
    }
    __syncthreads();
    if (threadIdx.x == 0 && s_live) s_base = (u32)atomicAdd(&ctr[CTR_NCONE], (u64)s_live);
    __syncthreads();
    if (sides) {
        u32 o = s_base + (u32)rank;
        if (sides & 1) cone_list[o++] = ((u32)v << 1);
        if (sides & 2) cone_list[o] = ((u32)v << 1) | 1u;
    }
    if (threadIdx.x < 5 && s_cnt[threadIdx.x]) atomicAdd(&ctr[CTR_V_POS + threadIdx.x], (u64)s_cnt[threadIdx.x]);
}

// ---------------------------------------------------------------------------------------
// host driver
// ---------------------------------------------------------------------------------------
// Work forked onto the vertex stream must not outlive an early (error) return: the temporaries it reads are
// released on `st` by TmpPool, and sdf_destroy never sees that stream.  Declared AFTER the TmpPool it protects,
// so it is destroyed (and the stream drained) first.
struct StreamDrain {
    cudaStream_t s; bool armed;
    StreamDrain() : s(nullptr), armed(false) {}
    ~StreamDrain() { if (armed) cudaStreamSynchronize(s); }
};

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

static u32 pow2_at_least(u64 n) {
    u64 c = 64;
    while (c < n) c <<= 1;
    return (u32)c;
}

// error path: which of NOTCLOSED / ORIENT does the invalid edge table amount to?
static int classify_edge_errors(sdf_mesh *m, int nc, TmpPool &tmp, cudaStream_t st) {
    if (nc & 1) {
        int f = ERRB_NOTCLOSED;
        CK(cudaMemcpyAsync(m->d_flags, &f, sizeof(int), cudaMemcpyHostToDevice, st));
        return SDF_OK;
    }
    u64 *eka, *ekb, *scan_ws;
    u32 *va, *vb, *hist;
    CKS(tmp.get((void **)&eka, sizeof(u64) * nc));
    CKS(tmp.get((void **)&ekb, sizeof(u64) * nc));
    CKS(tmp.get((void **)&va, sizeof(u32) * nc));
    CKS(tmp.get((void **)&vb, sizeof(u32) * nc));
    CKS(tmp.get((void **)&hist, sizeof(u32) * radix_hist_elems(nc)));
    CKS(tmp.get((void **)&scan_ws, sizeof(u64) * scan_ws_elems((int64_t)radix_hist_elems(nc))));
    KL; edge_keys_kernel<<<blocks_for(nc), FB, 0, st>>>(m->cvid, nc, eka, va);
    int shifts[8];
    for (int p = 0; p < 8; p++) shifts[p] = 8 * p;
    bool first;
    CKS(radix_sort_pairs<u64>(eka, va, ekb, vb, nc, shifts, 8, hist, scan_ws, st, &first));
    KL; edge_validate_kernel<<<blocks_for(nc), FB, 0, st>>>(first ? eka : ekb, first ? va : vb, nc, m->cvid, m->d_flags);
    CK(cudaGetLastError());
    return SDF_OK;
}

// the library's second and third stream (vertex stage and hoisted A6a beside the edge stage): forked from st, drained
// on early returns
static int fork_vertex_stream(sdf_mesh *m, cudaStream_t st, cudaStream_t *vs_out, StreamDrain &drain,
                              cudaStream_t *bs_out = nullptr, StreamDrain *bdrain = nullptr) {
    *vs_out = st;
    if (bs_out) *bs_out = st;
    const char *cf = getenv("SDF_CREATE_FORK");
    if (cf && cf[0] == '0') return SDF_OK;
    static cudaStream_t g_vs = nullptr, g_bs = nullptr;
    static int g_vs_dev = -1;
    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (!g_vs || g_vs_dev != dev) {
        CK(cudaStreamCreateWithFlags(&g_vs, cudaStreamNonBlocking));
        CK(cudaStreamCreateWithFlags(&g_bs, cudaStreamNonBlocking));
        g_vs_dev = dev;
    }
    CKS(ev_get(m, &m->ev_fork));
    CKS(ev_get(m, &m->ev_join));
    CK(cudaEventRecord(m->ev_fork, st));
    CK(cudaStreamWaitEvent(g_vs, m->ev_fork, 0));
    drain.s = g_vs; drain.armed = true;
    *vs_out = g_vs;
    if (bs_out && bdrain && m->hoist_g) {
        CKS(ev_get(m, &m->ev_bjoin));
        CK(cudaStreamWaitEvent(g_bs, m->ev_fork, 0));
        bdrain->s = g_bs; bdrain->armed = true;
        *bs_out = g_bs;
    }
    return SDF_OK;
}

// the one host crossing of sdf_create: validation flags, vertex / wedge / cone counts, class counters (and, inside
// sdf_transform, the brick total of the hoisted A6a)
static int finish_features(sdf_mesh *m, int nc, int vcap, TmpPool &tmp, cudaStream_t st) {
    int hflags[4] = {0, 0, 0, 0};
    {
        // counters and flags are adjacent in the slab: one copy
        const size_t span = (size_t)((char *)(m->d_flags + 4) - (char *)m->d_ctr);
        u64 both[CTR_TOTAL + 64];
        if (span <= sizeof(both) && (char *)m->d_flags > (char *)m->d_ctr) {
            CK(cudaMemcpyAsync(both, m->d_ctr, span, cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            memcpy(m->h_ctr, both, sizeof(u64) * CTR_COUNT);
            memcpy(hflags, (char *)both + ((char *)m->d_flags - (char *)m->d_ctr), sizeof(hflags));
        } else {
            CK(cudaMemcpyAsync(hflags, m->d_flags, sizeof(hflags), cudaMemcpyDeviceToHost, st));
            CK(cudaMemcpyAsync(m->h_ctr, m->d_ctr, sizeof(u64) * CTR_COUNT, cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
        }
    }
    int status = status_from_flags(hflags[0]);
    m->V = (int64_t)(m->h_ctr[CTR_V] < (u64)vcap ? m->h_ctr[CTR_V] : (u64)vcap);
    m->Elive = (int64_t)m->h_ctr[CTR_ELIVE];
    m->NC = (int64_t)m->h_ctr[CTR_NCONE];
    // closed + consistently oriented <=> every half-edge was claimed into a pair
    const u64 pairs = m->h_ctr[CTR_E_CONVEX] + m->h_ctr[CTR_E_CONCAVE] + m->h_ctr[CTR_E_FLAT];
    if ((status == SDF_OK || status == SDF_ENOTCLOSED) && 2 * pairs != (u64)nc) {
        // which of "not closed" / "mis-oriented" it is: the exact (sorted-key) classifier
        CKS(classify_edge_errors(m, nc, tmp, st));
        CK(cudaMemcpyAsync(hflags, m->d_flags, sizeof(hflags), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        status = status_from_flags(hflags[0]);
        if (status == SDF_OK) status = SDF_ENOTCLOSED;
    }
    return status;
}

// A0: order the triangles along a Morton curve, fine enough that consecutive triangles share vertices and edges
// (every later gather / scatter then stays L2-local; the paper sorts by Morton code for the same reason,
// PAPER.md:296-332): bins per axis ~ sqrt(F / 192) -- a surface occupies ~6 n^2 of the n^3 bins, ~32 triangles each.
// One-pass counting sort (fine_bin_kernel).  The order is internal: ids written to the output are the caller's.
struct OrderWs { u32 *cnt, *key, *ticket; u64 *scan_ws; int *bbox; int bits; int64_t nbins; bool on; };
static void order_plan(int64_t F, int64_t min_f, OrderWs *w) {
    const char *nb = getenv("SDF_NO_BINNING");
    w->on = !(nb && nb[0] == '1') && F >= min_f;
    int bits = 2;
    while (bits < 7 && (int64_t)192 * (1 << (2 * bits)) < F) bits++;
    if (const char *bb = getenv("SDF_BIN_BITS")) { const int v = atoi(bb); if (v >= 1 && v <= 8) bits = v; }
    w->bits = bits;
    w->nbins = (int64_t)1 << (3 * bits);
}
static void order_carve(Carver &c, int64_t F, OrderWs *w) {
    if (!w->on) return;
    w->cnt = c.take<u32>((size_t)w->nbins);
    w->scan_ws = c.take<u64>(scan_ws_elems(w->nbins));
    w->key = c.take<u32>((size_t)F); w->ticket = c.take<u32>((size_t)F);
    w->bbox = c.take<int>(8);
}
static int order_triangles(const float *src, int64_t F, const OrderWs &w, u32 *perm, cudaStream_t st) {
    if (!w.on) {
        KL; identity_perm_kernel<<<blocks_for(F), FB, 0, st>>>((int)F, perm);
        return SDF_OK;
    }
    const int lo_hi[8] = {0x7FFFFFFF, 0x7FFFFFFF, 0x7FFFFFFF, (int)0x80000000, (int)0x80000000, (int)0x80000000, 0, 0};
    CK(cudaMemcpyAsync(w.bbox, lo_hi, sizeof(lo_hi), cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(w.cnt, 0, sizeof(u32) * (size_t)w.nbins, st));
    const int stride = F > (1 << 20) ? 64 : (F > (1 << 16) ? 8 : 1);
    KL; bbox_sample_kernel<<<blocks_for((F + stride - 1) / stride), FB, 0, st>>>(src, (int)F, stride, w.bbox);
    KL; fine_bin_kernel<<<blocks_for(F), FB, 0, st>>>(src, (int)F, w.bbox, w.bits, w.cnt, w.key, w.ticket);
    CKS(launch_scan(BinIn{w.cnt}, BinOut{w.cnt}, w.nbins, w.scan_ws, (u64 *)nullptr, st));
    KL; fine_scatter_kernel<<<blocks_for(F), FB, 0, st>>>((int)F, w.cnt, w.key, w.ticket, perm);
    CK(cudaGetLastError());
    return SDF_OK;
}

static int build_features_global(sdf_mesh *m, const float *tri, int on_device, cudaStream_t st) {
    const int64_t F = m->F;
    const int nc = (int)(3 * F);
    const sdf_allocator *al = &m->alloc;
    TmpPool tmp(al, st);
    StreamDrain drain, bdrain;
    m->E = nc / 2;
    // every vertex of a closed surface has at least two corners, so V <= 3F/2; the per-vertex tables are sized by that
    // bound (no host crossing for the count) and a soup with more vertices is flagged not closed by ingest_weld_kernel
    const int vcap = (int)((3 * F < 3 * F / 2 + 64) ? 3 * F : 3 * F / 2 + 64);
    m->V = vcap;                                   // provisional: the count comes back with the validation flags

    // persistent tables: one slab
    for (int pass = 0; pass < 2; pass++) {
        Carver c(m->slab_f);
        m->soup = c.take<float>(9 * (size_t)F);
        m->fn = c.take<float>(3 * (size_t)F);
        m->cvid = c.take<int>(3 * (size_t)F);
        m->adj = c.take<int>(3 * (size_t)F);
        m->erec = c.take<EdgeRec>((size_t)(m->E > 0 ? m->E : 1));
        m->fsm = c.take<float>((size_t)F);
        m->perm = c.take<int>((size_t)F);
        m->inv_perm = c.take<int>((size_t)F);
        m->vrec = c.take<VertexRec>((size_t)vcap);
        m->vmint = c.take<int>((size_t)vcap);
        m->cone_list = c.take<u32>(2 * (size_t)vcap);
        m->vsm = c.take<unsigned char>((size_t)vcap);
        m->d_ctr = c.take<u64>(CTR_TOTAL);
        m->d_flags = c.take<int>(4);
        m->fill_state = c.take<u32>(1024);                   // (small blocks of their own would each cost an allocator call)
        m->hoist_g_dev = c.take<GridParams>(1);
        if (pass == 0) CKS(dev_alloc(al, &m->slab_f, c.off, st));
    }
    CK(cudaMemsetAsync(m->d_ctr, 0, (size_t)((char *)(m->d_flags + 4) - (char *)m->d_ctr), st));      // counters and flags: adjacent

    // smooth features get no polyhedron of their own (common.cuh, SMOOTH_SIN_DEFAULT); SDF_SMOOTH_SIN=0 switches that off
    float smooth_sin = SMOOTH_SIN_DEFAULT;
    if (const char *ss = getenv("SDF_SMOOTH_SIN")) { smooth_sin = (float)atof(ss); if (!(smooth_sin >= 0.0f && smooth_sin <= SMOOTH_SIN_DEFAULT)) smooth_sin = SMOOTH_SIN_DEFAULT; }
    const char *rc = getenv("SDF_RUFF");
    const bool ruff_cone = rc && !strcmp(rc, "cone");

    // ---- A0 ingest + A1 weld (hash table on the exact coordinate bits)
    CKS(maybe_prefill(m, 1, st));
    stage_mark(m, SDF_T_INGEST_WELD, 0, st);
    const u32 capw = pow2_at_least((u64)nc + (u64)nc / 4 + 1);     // load <= 0.8 even if no vertex is shared
    const u32 cape = pow2_at_least((u64)nc + 1);                   // <= 3F/2 forward half-edges: load <= 0.5
    float *staging = nullptr;
    OrderWs ow = {};
    order_plan(F, 131072, &ow);                     // smaller meshes live in L2 anyway
    u32 *wtab = nullptr, *slot = nullptr, *etab = nullptr, *wvid = nullptr;
    int *vcorner = nullptr, *vside = nullptr;
    u64 *vacc = nullptr;
    double *vn64 = nullptr;
    long long *vcosq = nullptr, *vcospos = nullptr;
    void *tslab = nullptr;
    for (int pass = 0; pass < 2; pass++) {
        Carver c(tslab);
        wtab = c.take<u32>((size_t)capw);           // wtab and etab adjacent: one memset
        etab = c.take<u32>((size_t)cape);
        wvid = c.take<u32>((size_t)capw);           // slot -> vertex id, written by the inserter (no reset needed)
        slot = c.take<u32>((size_t)nc);
        vcorner = c.take<int>((size_t)vcap);
        vacc = c.take<u64>(3 * (size_t)vcap);
        vside = c.take<int>((size_t)vcap);
        vcosq = c.take<long long>((size_t)vcap);
        if (ruff_cone) vcospos = c.take<long long>((size_t)vcap);
        vn64 = c.take<double>(3 * (size_t)vcap);
        if (!on_device) staging = c.take<float>(9 * (size_t)F);
        order_carve(c, F, &ow);
        if (pass == 0) CKS(tmp.get(&tslab, c.off));
    }
    const float *src = tri;
    if (!on_device) {
        CK(cudaMemcpyAsync(staging, tri, sizeof(float) * 9 * F, cudaMemcpyHostToDevice, st));
        src = staging;
    }
    // the table resets (0.2 GB at C4) run on the second stream beside the latency-bound ordering kernels
    {
        cudaStream_t ms = st;
        StreamDrain mdrain;
        if (ow.on) CKS(fork_vertex_stream(m, st, &ms, mdrain));        // (small meshes: the fork costs more than it hides)
        CK(cudaMemsetAsync(wtab, 0xFF, (size_t)((char *)(etab + cape) - (char *)wtab), ms));
        if (ow.on) CKS(order_triangles(src, F, ow, (u32 *)m->perm, st));      // (not sorted: ingest_weld_kernel fills the identity)
        if (ms != st) {
            CK(cudaEventRecord(m->ev_join, ms));
            CK(cudaStreamWaitEvent(st, m->ev_join, 0));
            mdrain.armed = false;
        }
    }
    WeldTab wt = {wtab, capw - 1, 0u, ow.cnt, ow.bbox, ow.bits, (u32)F};
    {
        const char *ul = getenv("SDF_UNIFORM_TABLES");
        if (ow.on && !(ul && ul[0] == '1') && capw >= 4096) wt.scale = (u32)((((u64)capw - 1024) << 12) / (u64)F);
    }
    KL; ingest_weld_kernel<<<blocks_for(nc), FB, 0, st>>>(src, ow.on ? m->perm : nullptr, nc, m->soup, m->inv_perm, wt, slot, wvid, vcorner,
                                                        vacc, vcosq, vcospos, vside, m->vmint, vcap, m->d_ctr, m->d_flags, m->perm);
    stage_mark(m, SDF_T_INGEST_WELD, 1, st);

    // ---- A3 (per triangle), A2 edge table
    CKS(maybe_prefill(m, 2, st));
    stage_mark(m, SDF_T_EDGES, 0, st);
    // sdf_transform: A6a's workspace is taken in the order of `st` before anything touches it; tri_geom_kernel then marks
    // the bricks as it goes and the vertex stream only runs the scan
    const GridParams *mark_g = nullptr;
    unsigned char *mark_flag = nullptr;
    if (F >= ((int64_t)1 << 21)) CKS(maybe_begin_bricks(m, st, &mark_g, &mark_flag));   // (big triangles mark hundreds of bricks per thread: C5 loses 0.14 ms)
    else CKS(maybe_alloc_brick_ws(m, st));
    KL; tri_geom_kernel<<<blocks_for(F), FB, 0, st>>>(m->soup, wvid, slot, (int)F, m->cvid, m->fn, vacc, etab, cape - 1, m->d_flags,
                                                    mark_g, mark_flag, m->adj, m->fsm);
    // the vertex stage needs only what tri_geom wrote: it runs on a second stream beside the edge stage
    // (and A6a -- brick marks unless tri_geom made them, scan -- on a third one: it needs the soup and the normals only)
    cudaStream_t vs = st, bs = st;
    CKS(fork_vertex_stream(m, st, &vs, drain, &bs, &bdrain));
    CKS(maybe_prefill(m, 3, st));
    // pairing, classes and wedge records in one pass
    KL; edge_pair_record_kernel<<<blocks_for(F), FB, 0, st>>>(m->cvid, (int)F, etab, cape - 1, m->adj, m->soup, m->fn, m->perm,
                                                            smooth_sin, m->erec, (int)m->E, (int *)m->fsm, m->d_ctr, m->d_flags);
    CKS(maybe_prepare_bricks(m, st, bs, mark_g != nullptr));
    if (bs != st) CK(cudaEventRecord(m->ev_bjoin, bs));
    CK(cudaGetLastError());
    stage_mark(m, SDF_T_EDGES, 1, st);

    // ---- A3/A4 vertices (garbage-in on invalid input is harmless: ids stay in range)
    stage_mark(m, SDF_T_VERTICES, 0, vs);
    KL; vertex_normal_kernel<<<blocks_for(vcap), FB, 0, vs>>>(vacc, vcap, m->d_ctr + CTR_V, vn64);
    KL; vertex_cone_kernel<<<blocks_for(F), FB, 0, vs>>>(m->soup, m->cvid, (int)F, vn64, vcosq, vside, m->perm, m->vmint, vcospos);
    KL; vertex_record_kernel<<<blocks_for(vcap), FB, 0, vs>>>(m->soup, vcorner, vn64, nullptr, m->d_ctr + CTR_V, vcosq, vside, vcap,
                                                           vcospos, smooth_sin, m->vrec, m->vsm, m->cone_list, m->d_ctr);
    CK(cudaGetLastError());
    stage_mark(m, SDF_T_VERTICES, 1, vs);
    if (bs != st) {
        CK(cudaStreamWaitEvent(st, m->ev_bjoin, 0));
        bdrain.armed = false;
    }
    if (vs != st) {
        CK(cudaEventRecord(m->ev_join, vs));
        CK(cudaStreamWaitEvent(st, m->ev_join, 0));
        drain.armed = false;           // joined: `st` now carries the dependency
    }
    // sdf_transform: the sentinel fill starts as soon as the feature kernels have drained, under the host crossing
    CKS(maybe_prefill(m, 4, st));
    return finish_features(m, nc, vcap, tmp, st);
}

// ===================================================================================================
// the tile-local builder (SDF_BUILDER=tile, an ablation; tile_features.cuh)
// ===================================================================================================
static int build_features_tile(sdf_mesh *m, const float *tri, int on_device, cudaStream_t st) {
    const int64_t F = m->F;
    const int nc = (int)(3 * F);
    const sdf_allocator *al = &m->alloc;
    TmpPool tmp(al, st);
    StreamDrain drain;
    m->E = nc / 2;
    // every vertex of a closed surface has at least two corners, so V <= 3F/2; the per-vertex tables are sized by that
    // bound (no host crossing for the count) and a soup with more vertices is flagged not closed by tile_weld_kernel
    const int vcap = (int)((3 * F < 3 * F / 2 + 64) ? 3 * F : 3 * F / 2 + 64);
    m->V = vcap;                                   // provisional: the count comes back with the validation flags
    const int ntiles = (int)((F + TT - 1) / TT);

    for (int pass = 0; pass < 2; pass++) {
        Carver c(m->slab_f);
        m->soup = c.take<float>(9 * (size_t)F);
        m->fn = c.take<float>(3 * (size_t)F);
        m->cvid = c.take<int>(3 * (size_t)F);
        m->adj = c.take<int>(3 * (size_t)F);
        m->erec = c.take<EdgeRec>((size_t)(m->E > 0 ? m->E : 1));
        m->fsm = c.take<float>((size_t)F);
        m->perm = c.take<int>((size_t)F);
        m->inv_perm = c.take<int>((size_t)F);
        m->vrec = c.take<VertexRec>((size_t)vcap);
        m->vmint = c.take<int>((size_t)vcap);
        m->cone_list = c.take<u32>(2 * (size_t)vcap);
        m->vsm = c.take<unsigned char>((size_t)vcap);
        m->d_ctr = c.take<u64>(CTR_TOTAL);
        m->d_flags = c.take<int>(4);
        m->fill_state = c.take<u32>(1024);                   // (small blocks of their own would each cost an allocator call)
        m->hoist_g_dev = c.take<GridParams>(1);
        if (pass == 0) CKS(dev_alloc(al, &m->slab_f, c.off, st));
    }
    CK(cudaMemsetAsync(m->d_ctr, 0, sizeof(u64) * CTR_TOTAL, st));
    CK(cudaMemsetAsync(m->d_flags, 0, sizeof(int) * 4, st));

    float smooth_sin = SMOOTH_SIN_DEFAULT;
    if (const char *ss = getenv("SDF_SMOOTH_SIN")) { smooth_sin = (float)atof(ss); if (!(smooth_sin >= 0.0f && smooth_sin <= SMOOTH_SIN_DEFAULT)) smooth_sin = SMOOTH_SIN_DEFAULT; }
    const char *rc = getenv("SDF_RUFF");
    const bool ruff_cone = rc && !strcmp(rc, "cone");

    CKS(maybe_prefill(m, 1, st));
    stage_mark(m, SDF_T_INGEST_WELD, 0, st);
    // global tables: only the unique vertices of each tile and the half-edges without a partner in their tile go
    // through them, but a hostile soup can still send every corner there: sized for that, so no probe loop can fill one
    const u32 capw = pow2_at_least((u64)nc + (u64)nc / 4 + 1);
    const u32 cape = pow2_at_least((u64)nc + 1);
    float *staging = nullptr;
    OrderWs ow = {};
    order_plan(F, 4 * TT, &ow);                     // a few tiles need no order
    u32 *wtab = nullptr, *etab = nullptr;
    int *vcorner = nullptr, *vside = nullptr;
    u64 *vacc = nullptr;
    long long *vcosq = nullptr, *vcospos = nullptr;
    TileTables tt = {nullptr, nullptr, nullptr, nullptr};
    void *tslab = nullptr;
    for (int pass = 0; pass < 2; pass++) {
        Carver c(tslab);
        wtab = c.take<u32>((size_t)capw);           // wtab and etab adjacent: one memset
        etab = c.take<u32>((size_t)cape);
        tt.wvid = c.take<u32>((size_t)capw);
        tt.clv = c.take<unsigned short>((size_t)nc);
        tt.tvid = c.take<u32>((size_t)nc);
        tt.tnlv = c.take<int>((size_t)ntiles);
        vcorner = c.take<int>((size_t)vcap);
        vacc = c.take<u64>(3 * (size_t)vcap);
        vside = c.take<int>((size_t)vcap);
        vcosq = c.take<long long>((size_t)vcap);
        if (ruff_cone) vcospos = c.take<long long>((size_t)vcap);
        if (!on_device) staging = c.take<float>(9 * (size_t)F);
        order_carve(c, F, &ow);
        if (pass == 0) CKS(tmp.get(&tslab, c.off));
    }
    const float *src = tri;
    if (!on_device) {
        CK(cudaMemcpyAsync(staging, tri, sizeof(float) * 9 * F, cudaMemcpyHostToDevice, st));
        src = staging;
    }
    CK(cudaMemsetAsync(wtab, 0xFF, (size_t)((char *)(etab + cape) - (char *)wtab), st));
    CKS(order_triangles(src, F, ow, (u32 *)m->perm, st));
    // (per call: the attribute belongs to the current device, and the two calls cost a few microseconds)
    CK(cudaFuncSetAttribute(tile_geom_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TileGeomSmem)));
    CK(cudaFuncSetAttribute(tile_cone_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(TileConeSmem)));
    // A1: weld inside the tiles, the tiles' unique vertices through the global table
    KL; tile_weld_kernel<<<ntiles, TB, 0, st>>>(src, m->perm, (int)F, m->soup, m->inv_perm, wtab, capw - 1, tt, vcorner, vacc,
                                              vcosq, vcospos, vside, m->vmint, vcap, m->d_ctr, m->d_flags);
    stage_mark(m, SDF_T_INGEST_WELD, 1, st);
    // A2 + A3: ids, normals, angle-weighted sums, edges inside the tiles
    CKS(maybe_prefill(m, 2, st));
    stage_mark(m, SDF_T_EDGES, 0, st);
    KL; tile_geom_kernel<<<ntiles, TB, sizeof(TileGeomSmem), st>>>(m->soup, (int)F, m->perm, tt, wtab, m->cvid, m->fn, vacc, m->adj,
                                                                 etab, cape - 1, smooth_sin, m->erec, (int)m->E, m->fsm,
                                                                 m->d_ctr, m->d_flags);
    CK(cudaGetLastError());
    // sdf_transform: the workspace of A6a is taken in the order of `st` BEFORE the fork (the vertex stream touches it first)
    CKS(maybe_alloc_brick_ws(m, st));
    cudaStream_t vs = st;
    CKS(fork_vertex_stream(m, st, &vs, drain));
    CKS(maybe_prefill(m, 3, st));
    // edges across tile boundaries
    KL; edge_pair_record_kernel<<<blocks_for(F), FB, 0, st>>>(m->cvid, (int)F, etab, cape - 1, m->adj, m->soup, m->fn, m->perm,
                                                            smooth_sin, m->erec, (int)m->E, (int *)m->fsm, m->d_ctr, m->d_flags);
    CK(cudaGetLastError());
    stage_mark(m, SDF_T_EDGES, 1, st);
    // A3/A4 vertices: cone angles, sides, lowest triangle ids per tile; then the records
    stage_mark(m, SDF_T_VERTICES, 0, vs);
    KL; tile_cone_kernel<<<ntiles, TB, sizeof(TileConeSmem), vs>>>(m->soup, (int)F, m->perm, tt, vacc, vcosq, vside, m->vmint, vcospos);
    KL; vertex_record_kernel<<<blocks_for(vcap), FB, 0, vs>>>(m->soup, vcorner, nullptr, vacc, m->d_ctr + CTR_V, vcosq, vside, vcap,
                                                           vcospos, smooth_sin, m->vrec, m->vsm, m->cone_list, m->d_ctr);
    CK(cudaGetLastError());
    stage_mark(m, SDF_T_VERTICES, 1, vs);
    CKS(maybe_prepare_bricks(m, st, vs, false));
    if (vs != st) {
        CK(cudaEventRecord(m->ev_join, vs));
        CK(cudaStreamWaitEvent(st, m->ev_join, 0));
        drain.armed = false;           // joined: `st` now carries the dependency
    }
    // sdf_transform: the sentinel fill starts as soon as the feature kernels have drained, under the host crossing
    CKS(maybe_prefill(m, 4, st));
    return finish_features(m, nc, vcap, tmp, st);
}

int build_features(sdf_mesh *m, const float *tri, int on_device, cudaStream_t st) {
    // SDF_BUILDER=tile: the tile-local builder (tile_features.cuh), measured slower on a B200: an ablation
    const char *b = getenv("SDF_BUILDER");
    if (b && !strcmp(b, "tile")) return build_features_tile(m, tri, on_device, st);
    return build_features_global(m, tri, on_device, st);
}
