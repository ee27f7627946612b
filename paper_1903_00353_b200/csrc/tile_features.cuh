// tile_features.cuh -- included by features.cu.  Holds (1) what both feature builders share: the edge classifier
// (edge_class_of), the record writer, edge_pair_record_kernel (pairing through the global half-edge table, class and
// wedge record in one pass -- the default builder runs it over every half-edge) and vertex_axis64; (2) the TILE-LOCAL
// builder, SDF_BUILDER=tile: an ablation, bit-identical to the default builder in every table and grid
// (tests/test_gpu_features.py) and measured slower on a B200 (C4 3.84 against 3.36 ms when the two were compared).
//
// The paper regroups the unordered STL entries with a Morton sort and a per-group serial pass and
// names that regrouping as its bottleneck.  The default builder (features.cu) welds vertices and
// pairs half-edges through hash tables in global memory: every one of the 3F corners costs several random L2 sectors
// (478 M sectors for 144 MB of input at C4, profiles/r2_atomics.md).  The tile-local builder was the attempt to keep
// that traffic on chip:
//
// The soup is put in a fine Morton order (the one-pass counting sort of features.cu) and cut into tiles of TT
// consecutive triangles.  Inside a tile everything happens in shared memory:
//   T1 tile_weld_kernel   gather + canonicalise the tile, weld its corners in a shared-memory hash table (exact bits),
//                         then only the tile's UNIQUE vertices (~1/4 of its corners) go through the global weld table
//                         (find-or-insert; the inserter takes a vertex id from a counter and resets the accumulators)
//   T3 tile_geom_kernel   vertex ids of the corners, fp64 face normals and corner angles, the angle-weighted normal
//                         sums (eq.8) combined per tile vertex in shared memory (32-bit limbs) and added
//                         to the global accumulators once per tile vertex; half-edges paired inside the tile, their
//                         edge classes and wedge records written; only half-edges without a partner in
//                         the tile (patch boundary) enter the global half-edge table
//   T4 edge_pair_record_kernel   the boundary half-edges: pairing through the global table, class + record in one pass
//   T5 tile_cone_kernel   cone angle (eq.9), side bits and lowest triangle id,
//                         combined per tile vertex in shared memory, one global atomic each per tile vertex
// It halves the L2 sectors (223 M) and loses on instructions and occupancy: 44-69 KB of shared memory and 76-80 registers
// per thread, 300 M warp instructions in tile_geom_kernel alone; and a run of a space-filling curve is several patches,
// not one: 54 % of a tile's vertices also occur in another tile.
// Vertex ids and the order of the edge records depend on the order in which blocks run (both builders); nothing that
// reaches the output does (ids written to the grids are the caller's triangle ids, all sums are integer).
#pragma once

#define TT 512                 // triangles per tile
#define TC (3 * TT)            // corners per tile
#define TB 256                 // threads per block of the tile kernels
#define TCPT (TC / TB)         // corners per thread
#define TLH 4096               // slots of the shared-memory hash tables (load <= 0.375)
#define TCAP 768               // tile vertices with shared-memory accumulators (the others fall back to global atomics)
#define SHARED_BIT 0x80000000u // weld table slot: the vertex was found by a tile other than the one that inserted it
#define LIMB_BITS 21
#define LIMB_MASK 0x1FFFFFu

struct TileTables {
    unsigned short *clv;       // [3F] corner -> index of its vertex among the unique vertices of its tile
    u32 *tvid;                 // [3F] (tile, tile vertex): T1 weld-table slot; T3 on: vertex id | SHARED_BIT
    int *tnlv;                 // [tiles] unique vertices of the tile
    u32 *wvid;                 // [weld table size] slot -> vertex id (written by the inserter)
};

// block-wide exclusive scan of one small count per thread (TB threads); total returned in *total
__device__ __forceinline__ int tile_excl_scan(int v, u32 *s_w, int *total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_w[w] = (u32)inc;
    __syncthreads();
    int base = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < TB / 32; i++) {
        const int x = (int)s_w[i];
        if (i < w) base += x;
        tot += x;
    }
    __syncthreads();
    *total = tot;
    return base + inc - v;
}

// -------------------------------------------------------------------------------------------------------------
// T1: gather, canonicalise, local weld, global find-or-insert of the tile's unique vertices
// -------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(TB) tile_weld_kernel(const float *__restrict__ in, const int *__restrict__ perm, int F,
                                                       float *__restrict__ soup, int *__restrict__ inv_perm, u32 *wtab,
                                                       u32 wmask, TileTables tt, int *__restrict__ vcorner,
                                                       u64 *__restrict__ vacc, long long *__restrict__ vcosq,
                                                       long long *__restrict__ vcospos, int *__restrict__ vside,
                                                       int *__restrict__ vmint, int vcap, u64 *ctr, int *flags) {
    __shared__ u32 s_pos[TC * 3];
    __shared__ u32 s_lh[TLH];
    __shared__ unsigned short s_hs[TC], s_lv[TC], s_headc[TC];
    __shared__ u32 s_w[TB / 32];
    __shared__ u32 s_nins, s_vbase;
    const int tid = threadIdx.x;
    const int b0 = blockIdx.x * TT;
    const int nt = min(TT, F - b0), nc = 3 * nt;
    if (tid == 0) s_nins = 0;
    for (int j = tid; j < TLH; j += TB) s_lh[j] = EMPTY32;
    bool bad = false;
    // gather: float j of the tile is component j % 9 of tile triangle j / 9, so consecutive lanes read consecutive
    // floats of one triangle (36 contiguous bytes per 9 lanes instead of 32 different sectors per load)
    for (int j = tid; j < 9 * nt; j += TB) {
        const int i = j / 9, k = j - 9 * i;
        const int t = perm[b0 + i];
        const float x = in[9 * (size_t)t + k];
        if (!isfinite(x)) bad = true;
        s_pos[j] = __float_as_uint(x + 0.0f);                        // -0 + +0 = +0
        if (k == 0) inv_perm[t] = b0 + i;
    }
    if (bad) atomicOr(flags, ERRB_NONFINITE);
    __syncthreads();
    for (int j = tid; j < 9 * nt; j += TB) soup[9 * (size_t)b0 + j] = __uint_as_float(s_pos[j]);

    // ---- weld inside the tile: a slot holds a corner of its vertex and converges to the lowest one
    for (int c = tid; c < nc; c += TB) {
        const u32 x = s_pos[3 * c], y = s_pos[3 * c + 1], z = s_pos[3 * c + 2];
        u32 h = mix32(x, y, z) & (TLH - 1);
        for (;;) {
            u32 cur = ((volatile u32 *)s_lh)[h];
            if (cur == EMPTY32) {
                cur = atomicCAS(&s_lh[h], EMPTY32, (u32)c);
                if (cur == EMPTY32) break;
            }
            if (s_pos[3 * cur] == x && s_pos[3 * cur + 1] == y && s_pos[3 * cur + 2] == z) {
                if ((u32)c < cur) atomicMin(&s_lh[h], (u32)c);
                break;
            }
            h = (h + 1) & (TLH - 1);
        }
        s_hs[c] = (unsigned short)h;
    }
    __syncthreads();
    // ---- number the tile's vertices in the order of their lowest corners
    u32 hm = 0;
    int cnt = 0;
#pragma unroll
    for (int j = 0; j < TCPT; j++) {
        const int c = tid * TCPT + j;
        if (c < nc && s_lh[s_hs[c]] == (u32)c) { hm |= 1u << j; cnt++; }
    }
    int nlv;
    int o = tile_excl_scan(cnt, s_w, &nlv);
#pragma unroll
    for (int j = 0; j < TCPT; j++)
        if ((hm >> j) & 1u) {
            const int c = tid * TCPT + j;
            s_lv[c] = (unsigned short)o;
            s_headc[o] = (unsigned short)c;
            o++;
        }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < TCPT; j++) {
        const int c = tid * TCPT + j;
        if (c < nc && !((hm >> j) & 1u)) s_lv[c] = s_lv[s_lh[s_hs[c]]];
    }
    __syncthreads();
    for (int c = tid; c < nc; c += TB) tt.clv[3 * (size_t)b0 + c] = s_lv[c];
    if (tid == 0) tt.tnlv[blockIdx.x] = nlv;

    // ---- the tile's unique vertices through the global weld table.  A slot holds a corner (index in the internal
    // order) of its vertex; identity is checked on the exact bits of that corner in the immutable input
    u32 myslot[TCPT];
    int myrank[TCPT];
#pragma unroll
    for (int q = 0; q < TCPT; q++) {
        const int lv = tid + q * TB;
        myrank[q] = -1;
        myslot[q] = 0;
        if (lv >= nlv) continue;
        const int c = s_headc[lv];
        const u32 g = 3u * (u32)b0 + (u32)c;
        const u32 x = s_pos[3 * c], y = s_pos[3 * c + 1], z = s_pos[3 * c + 2];
        u32 h = mix32(x, y, z) & wmask;
        for (;;) {
            u32 cur = __ldcg(wtab + h);
            if (cur == EMPTY32) {
                cur = atomicCAS(wtab + h, EMPTY32, g);
                if (cur == EMPTY32) { myrank[q] = (int)atomicAdd(&s_nins, 1u); break; }
            }
            const u32 gc = cur & ~SHARED_BIT;
            const u32 ci = gc / 3u, ck = gc - 3u * ci;
            const float *qq = in + 9 * (size_t)perm[ci] + 3 * ck;
            if (canon_bits(qq[0]) == x && canon_bits(qq[1]) == y && canon_bits(qq[2]) == z) {
                if (!(cur & SHARED_BIT)) atomicOr(wtab + h, SHARED_BIT);
                break;
            }
            h = (h + 1) & wmask;
        }
        myslot[q] = h;
        tt.tvid[3 * (size_t)b0 + lv] = h;
    }
    __syncthreads();
    if (tid == 0 && s_nins) s_vbase = (u32)atomicAdd(&ctr[CTR_V], (u64)s_nins);
    __syncthreads();
#pragma unroll
    for (int q = 0; q < TCPT; q++) {
        if (myrank[q] < 0) continue;
        const int lv = tid + q * TB;
        u32 vid = s_vbase + (u32)myrank[q];
        if (vid >= (u32)vcap) {
            // more vertices than a closed surface of F triangles can have (every vertex of a closed surface has at
            // least two corners: V <= 3F/2): the per-vertex tables are not that large
            atomicOr(flags, ERRB_NOTCLOSED);
            tt.wvid[myslot[q]] = (u32)(vcap - 1);
            continue;
        }
        tt.wvid[myslot[q]] = vid;
        vcorner[vid] = (int)(3u * (u32)b0 + (u32)s_headc[lv]);
        vacc[3 * (size_t)vid] = 0ull; vacc[3 * (size_t)vid + 1] = 0ull; vacc[3 * (size_t)vid + 2] = 0ull;
        vcosq[vid] = 0x7F7F7F7F7F7F7F7Fll;
        if (vcospos) vcospos[vid] = 0x7F7F7F7F7F7F7F7Fll;
        vside[vid] = 0;
        vmint[vid] = 0x7F7F7F7F;
    }
}

// -------------------------------------------------------------------------------------------------------------
// edge class + record (shared by T3, T4 and the global builder's edge_record_kernel)
// -------------------------------------------------------------------------------------------------------------
struct EdgeGeom { const float *A, *B, *N1, *N2; };
// canonical direction a -> b = ascending exact position bits, so the record (and the fp32 rounding of every distance
// evaluated from it) does not depend on the order of the triangles in the soup; n1 stays the normal of the triangle
// that traverses a -> b.  (A, B): end points as the FORWARD half-edge's triangle (normal N1) traverses them.
__device__ __forceinline__ EdgeGeom edge_geom_of(const float *A, const float *B, const float *N1, const float *N2) {
    EdgeGeom g;
    g.A = A; g.B = B; g.N1 = N1; g.N2 = N2;
    const u32 *pa = (const u32 *)A, *pb = (const u32 *)B;
    if (pa[0] != pb[0] ? pa[0] > pb[0] : (pa[1] != pb[1] ? pa[1] > pb[1] : pa[2] > pb[2])) {
        g.A = B; g.B = A; g.N1 = N2; g.N2 = N1;
    }
    return g;
}
// PAPER.md:352 d = (ab x n1).n2 (normalised): +1 convex, -1 concave, 0 flat or smooth (then *smooth_bits holds the
// float bits of the margin sine, else 0), 2 knife
__device__ __forceinline__ int edge_class_of(const EdgeGeom &g, float smooth_sin, int *smooth_bits) {
    double ud[3], n1[3], n2[3], x[3];
#pragma unroll
    for (int i = 0; i < 3; i++) { ud[i] = (double)g.B[i] - (double)g.A[i]; n1[i] = g.N1[i]; n2[i] = g.N2[i]; }
    const double L = sqrt(ddot(ud, ud));
    dcross(ud, n1, x);
    const double d = (L > 0.0) ? ddot(x, n2) / L : 0.0;
    const double c12 = ddot(n1, n2);
    // flat: the wedge is thinner than 1e-6 * band and lies inside the eps-inflated neighbours (reading #5)
    int cl = d > 1e-6 ? 1 : (d < -1e-6 ? -1 : 0);
    // sin(dihedral) also vanishes when the faces fold back onto each other (n1 = -n2: a blade or a slit).  That edge
    // is as far from flat as an edge gets, and which side its wedge is on cannot be told from a vanishing
    // discriminant: class 2, "knife", whose extrusion is the whole cylinder about the edge
    if (cl == 0 && c12 <= 0.0) cl = 2;
    *smooth_bits = 0;
    // smooth: |sin| of the angle between the two normals below the threshold (and the angle acute).  No wedge; both
    // faces widen their prisms by reach * sin instead
    if (c12 > 0.0 && fabs(d) <= (double)smooth_sin) {
        *smooth_bits = __float_as_int(__double2float_ru(fabs(d) * 1.000001 + 1e-9));
        cl = 0;
    }
    return cl;
}
__device__ __forceinline__ void edge_record_write(EdgeRec *__restrict__ dst, const EdgeGeom &g, int tri, int cls) {
    EdgeRec r;
#pragma unroll
    for (int i = 0; i < 3; i++) { r.a[i] = g.A[i]; r.b[i] = g.B[i]; r.n1[i] = g.N1[i]; r.n2[i] = g.N2[i]; }
    r.tri = tri; r.cls = cls; r.pad[0] = r.pad[1] = 0;
    *dst = r;
}

// -------------------------------------------------------------------------------------------------------------
// T3: ids, geometry, normal sums, edges inside the tile
// -------------------------------------------------------------------------------------------------------------
struct TileGeomSmem {
    float pos[TC * 3];
    float fn[TT * 3];
    u32 vid[TC];
    int perm[TT];
    int fsm[TT];
    short ladj[TC];
    unsigned short lv[TC];
    union { u32 acc[TCAP * 9]; u32 eh[TLH]; } u;
    u32 w[TB / 32];
    u32 cnt[3];
    u32 live, base;
};

__global__ void __launch_bounds__(TB, 3) tile_geom_kernel(const float *__restrict__ soup, int F, const int *__restrict__ perm,
                                                          TileTables tt, const u32 *__restrict__ wtab,
                                                          int *__restrict__ cvid, float *__restrict__ fn,
                                                          u64 *__restrict__ vacc, int *__restrict__ adj, u32 *etab,
                                                          u32 emask, float smooth_sin, EdgeRec *__restrict__ erec, int E,
                                                          float *__restrict__ fsm, u64 *ctr, int *flags) {
    extern __shared__ __align__(16) unsigned char tile_smem[];
    TileGeomSmem &S = *(TileGeomSmem *)tile_smem;
    const int tid = threadIdx.x;
    const int b0 = blockIdx.x * TT;
    const int nt = min(TT, F - b0), nc = 3 * nt;
    const int nlv = tt.tnlv[blockIdx.x];
    const int nacc = min(nlv, TCAP);
    for (int j = tid; j < 9 * nt; j += TB) S.pos[j] = soup[9 * (size_t)b0 + j];
    for (int c = tid; c < nc; c += TB) { S.lv[c] = tt.clv[3 * (size_t)b0 + c]; S.ladj[c] = -1; }
    for (int i = tid; i < nt; i += TB) { S.perm[i] = perm[b0 + i]; S.fsm[i] = 0; }
    for (int lv = tid; lv < nlv; lv += TB) {
        const u32 h = tt.tvid[3 * (size_t)b0 + lv];
        const u32 v = tt.wvid[h] | (wtab[h] & SHARED_BIT);
        S.vid[lv] = v;
        tt.tvid[3 * (size_t)b0 + lv] = v;
    }
    for (int j = tid; j < nacc * 9; j += TB) S.u.acc[j] = 0;
    if (tid < 3) S.cnt[tid] = 0;
    if (tid == 3) S.live = 0;
    __syncthreads();
    for (int c = tid; c < nc; c += TB) cvid[3 * (size_t)b0 + c] = (int)(S.vid[S.lv[c]] & ~SHARED_BIT);

    // ---- per triangle: unit normal in fp64, corner angles, angle-weighted normal contributions (eq.8)
    for (int i = tid; i < nt; i += TB) {
        const int lv3[3] = {S.lv[3 * i], S.lv[3 * i + 1], S.lv[3 * i + 2]};
        double n[3], p[3][3];
        bool ok = tri_normal64(&S.pos[9 * i], n, p);
        if (!ok) {      // PAPER.md:137 "we disallow faces of zero area" (a repeated vertex is one, exactly)
            atomicOr(flags, ERRB_DEGENERATE);
            n[0] = n[1] = 0.0; n[2] = 1.0;
        }
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const float f = (float)n[j];
            S.fn[3 * i + j] = f;
            fn[3 * (size_t)(b0 + i) + j] = f;
        }
        if (!ok) continue;
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const int k1 = (k + 1) % 3, k2 = (k + 2) % 3;
            const double u[3] = {p[k1][0] - p[k][0], p[k1][1] - p[k][1], p[k1][2] - p[k][2]};
            const double w[3] = {p[k2][0] - p[k][0], p[k2][1] - p[k][1], p[k2][2] - p[k][2]};
            double x[3];
            dcross(u, w, x);
            const double alpha = atan2(sqrt(ddot(x, x)), ddot(u, w));          // corner angle, eq.8 weight
            const int lv = lv3[k];
#pragma unroll
            for (int a = 0; a < 3; a++) {
                // order-independent accumulation: 2^-40 fixed point, two's complement wrap-around.  In shared memory
                // the 64-bit value is split into 21-bit limbs (64-bit shared atomics are CAS loops, 32-bit ones are not):
                // a limb sum of at most 1536 corners stays below 2^32
                const long long v = llrint(alpha * n[a] * FIXSCALE);
                if (lv < TCAP) {
                    u32 *q = &S.u.acc[(lv * 3 + a) * 3];
                    const u32 l0 = (u32)((u64)v & LIMB_MASK), l1 = (u32)(((u64)v >> LIMB_BITS) & LIMB_MASK);
                    const int l2 = (int)(v >> (2 * LIMB_BITS));
                    if (l0) atomicAdd(q, l0);
                    if (l1) atomicAdd(q + 1, l1);
                    if (l2) atomicAdd(q + 2, (u32)l2);
                } else {
                    atomicAdd(&vacc[3 * (size_t)(S.vid[lv] & ~SHARED_BIT) + a], (u64)v);
                }
            }
        }
    }
    __syncthreads();
    for (int j = tid; j < nacc * 3; j += TB) {
        const u32 *q = &S.u.acc[j * 3];
        const u64 tot = (u64)q[0] + ((u64)q[1] << LIMB_BITS) + ((u64)(long long)(int)q[2] << (2 * LIMB_BITS));
        const int lv = j / 3, a = j - 3 * lv;
        if (tot) atomicAdd(&vacc[3 * (size_t)(S.vid[lv] & ~SHARED_BIT) + a], tot);
    }
    __syncthreads();

    // ---- half-edges inside the tile.  Half-edge c = 3i + k runs corner k -> k+1; "forward" here means
    // ascending tile vertex numbers.  Forward ones take the first empty slot on their probe path, backward ones look
    // the key up and claim it.  A pair both of whose end points also occur in other tiles is left to the global table:
    // only then can a third half-edge on the same two vertices exist outside the tile, and it must be seen.
    for (int j = tid; j < TLH; j += TB) S.u.eh[j] = EMPTY32;
    __syncthreads();
    for (int c = tid; c < nc; c += TB) {
        const u32 a = S.lv[c], b = S.lv[he_next(c)];
        if (a < b) {
            u32 h = edge_hash(a, b) & (TLH - 1);
            while (((volatile u32 *)S.u.eh)[h] != EMPTY32 || atomicCAS(&S.u.eh[h], EMPTY32, (u32)c) != EMPTY32) h = (h + 1) & (TLH - 1);
        }
    }
    __syncthreads();
    for (int c = tid; c < nc; c += TB) {
        const u32 a = S.lv[c], b = S.lv[he_next(c)];
        if (!(a > b)) continue;
        u32 h = edge_hash(b, a) & (TLH - 1);
        for (;;) {
            const u32 cur = ((volatile u32 *)S.u.eh)[h];
            if (cur == EMPTY32) break;                                   // no partner in this tile
            const int cand = (int)(cur & ~HE_MATCHED);
            if (S.lv[cand] == b && S.lv[he_next(cand)] == a) {
                if (S.vid[a] & S.vid[b] & SHARED_BIT) break;             // both end points shared: global table
                const u32 prev = atomicOr(&S.u.eh[h], HE_MATCHED);
                if (!(prev & HE_MATCHED)) { S.ladj[c] = (short)cand; S.ladj[cand] = (short)c; }
                else atomicOr(flags, ERRB_NOTCLOSED);                    // a third half-edge on this edge
                break;
            }
            h = (h + 1) & (TLH - 1);
        }
    }
    __syncthreads();
    // ---- adjacency out; half-edges without a partner here: the ascending ones (by vertex id) enter the global table
    for (int c = tid; c < nc; c += TB) {
        const int la = S.ladj[c];
        adj[3 * (size_t)b0 + c] = la >= 0 ? 3 * b0 + la : -1;
        if (la < 0) {
            const u32 u = S.vid[S.lv[c]] & ~SHARED_BIT, w = S.vid[S.lv[he_next(c)]] & ~SHARED_BIT;
            if (u < w) {
                u32 h = edge_hash(u, w) & emask;
                while (__ldcg(etab + h) != EMPTY32 || atomicCAS(etab + h, EMPTY32, (u32)(3 * b0 + c)) != EMPTY32) h = (h + 1) & emask;
            }
        }
    }
    // ---- class and record of the pairs made here (by the half-edge with ascending tile vertex numbers)
    int cls[TCPT], rank[TCPT];
#pragma unroll
    for (int q = 0; q < TCPT; q++) {
        const int c = tid + q * TB;
        cls[q] = 0; rank[q] = -1;
        if (c >= nc) continue;
        const int la = S.ladj[c];
        if (la < 0 || !(S.lv[c] < S.lv[he_next(c)])) continue;
        const int i = c / 3, i1 = la / 3;
        const EdgeGeom g = edge_geom_of(&S.pos[3 * c], &S.pos[3 * he_next(c)], &S.fn[3 * i], &S.fn[3 * i1]);
        int sb;
        const int cl = edge_class_of(g, smooth_sin, &sb);
        if (sb) { atomicMax(&S.fsm[i], sb); atomicMax(&S.fsm[i1], sb); }
        cls[q] = cl;
        atomicAdd(&S.cnt[cl > 0 ? 0 : (cl < 0 ? 1 : 2)], 1u);            // knife edges count as convex
        if (cl != 0) rank[q] = (int)atomicAdd(&S.live, 1u);
    }
    __syncthreads();
    if (tid == 0 && S.live) S.base = (u32)atomicAdd(&ctr[CTR_ELIVE], (u64)S.live);
    __syncthreads();
#pragma unroll
    for (int q = 0; q < TCPT; q++) {
        if (rank[q] < 0) continue;
        const u32 slot = S.base + (u32)rank[q];
        if (slot >= (u32)E) continue;            // cannot happen: pairs never outnumber 3F/2
        const int c = tid + q * TB, la = S.ladj[c], i = c / 3, i1 = la / 3;
        const EdgeGeom g = edge_geom_of(&S.pos[3 * c], &S.pos[3 * he_next(c)], &S.fn[3 * i], &S.fn[3 * i1]);
        const int x0 = S.perm[i], x1 = S.perm[i1];
        edge_record_write(erec + slot, g, x0 < x1 ? x0 : x1, cls[q]);
    }
    for (int i = tid; i < nt; i += TB) fsm[b0 + i] = __int_as_float(S.fsm[i]);
    if (tid < 3 && S.cnt[tid]) atomicAdd(&ctr[CTR_E_CONVEX + tid], (u64)S.cnt[tid]);
}

// -------------------------------------------------------------------------------------------------------------
// T4: half-edges without a partner in their tile.  One thread per triangle; its descending half-edges (by vertex
// id) look their partner up in the global table, claim it, and classify + record the edge at once.
// -------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(FB) edge_pair_record_kernel(const int *__restrict__ cvid, int F, u32 *etab, u32 mask,
                                                              int *adj, const float *__restrict__ soup,
                                                              const float *__restrict__ fn, const int *__restrict__ perm,
                                                              float smooth_sin, EdgeRec *__restrict__ erec, int E,
                                                              int *fsm_bits, u64 *ctr, int *flags) {
    __shared__ u32 s_cnt[3], s_live, s_base;
    if (threadIdx.x < 3) s_cnt[threadIdx.x] = 0;
    if (threadIdx.x == 3) s_live = 0;
    __syncthreads();
    const int t = blockIdx.x * FB + threadIdx.x;
    int part[3] = {-1, -1, -1}, cls[3] = {0, 0, 0}, rank[3] = {-1, -1, -1};
    if (t < F) {
        const u32 c[3] = {(u32)cvid[3 * (size_t)t], (u32)cvid[3 * (size_t)t + 1], (u32)cvid[3 * (size_t)t + 2]};
        u32 h[3];
        bool act[3];
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const u32 w = c[k], u = c[k == 2 ? 0 : k + 1];         // descending: w -> u with u < w
            act[k] = u < w && adj[3 * (size_t)t + k] < 0;
            h[k] = edge_hash(u, w) & mask;
        }
        while (act[0] || act[1] || act[2]) {
            u32 cur[3], ku[3], kw[3];
#pragma unroll
            for (int k = 0; k < 3; k++) cur[k] = act[k] ? __ldcg(etab + h[k]) : EMPTY32;
#pragma unroll
            for (int k = 0; k < 3; k++) {
                if (act[k] && cur[k] == EMPTY32) act[k] = false;             // no ascending partner
                if (act[k]) {
                    const int cand = (int)(cur[k] & ~HE_MATCHED);
                    ku[k] = (u32)cvid[cand]; kw[k] = (u32)cvid[he_next(cand)];
                }
            }
#pragma unroll
            for (int k = 0; k < 3; k++) {
                if (!act[k]) continue;
                const u32 w = c[k], u = c[k == 2 ? 0 : k + 1];
                if (ku[k] == u && kw[k] == w) {
                    const u32 prev = atomicOr(etab + h[k], HE_MATCHED);
                    if (!(prev & HE_MATCHED)) {
                        const int cand = (int)(cur[k] & ~HE_MATCHED);
                        adj[cand] = 3 * t + k;
                        adj[3 * t + k] = cand;
                        part[k] = cand;
                    } else atomicOr(flags, ERRB_NOTCLOSED);                 // a third half-edge on this edge
                    act[k] = false;
                } else {
                    h[k] = (h[k] + 1) & mask;
                }
            }
        }
#pragma unroll
        for (int k = 0; k < 3; k++) {
            if (part[k] < 0) continue;
            const int tf = part[k] / 3, kf = part[k] - 3 * tf;             // the ascending half-edge and its triangle
            const EdgeGeom g = edge_geom_of(soup + 9 * (size_t)tf + 3 * kf, soup + 9 * (size_t)tf + 3 * (kf == 2 ? 0 : kf + 1),
                                            fn + 3 * (size_t)tf, fn + 3 * (size_t)t);
            int sb;
            const int cl = edge_class_of(g, smooth_sin, &sb);
            if (sb) {
                if (fsm_bits[tf] < sb) atomicMax(&fsm_bits[tf], sb);
                if (fsm_bits[t] < sb) atomicMax(&fsm_bits[t], sb);
            }
            cls[k] = cl;
            atomicAdd(&s_cnt[cl > 0 ? 0 : (cl < 0 ? 1 : 2)], 1u);
            if (cl != 0) rank[k] = (int)atomicAdd(&s_live, 1u);
        }
    }
    __syncthreads();
    if (threadIdx.x == 0 && s_live) s_base = (u32)atomicAdd(&ctr[CTR_ELIVE], (u64)s_live);
    __syncthreads();
    if (t < F) {
#pragma unroll
        for (int k = 0; k < 3; k++) {
            if (rank[k] < 0) continue;
            const u32 slot = s_base + (u32)rank[k];
            if (slot >= (u32)E) continue;
            const int tf = part[k] / 3, kf = part[k] - 3 * tf;
            const EdgeGeom g = edge_geom_of(soup + 9 * (size_t)tf + 3 * kf, soup + 9 * (size_t)tf + 3 * (kf == 2 ? 0 : kf + 1),
                                            fn + 3 * (size_t)tf, fn + 3 * (size_t)t);
            const int x0 = perm[tf], x1 = perm[t];
            edge_record_write(erec + slot, g, x0 < x1 ? x0 : x1, cls[k]);
        }
    }
    if (threadIdx.x < 3 && s_cnt[threadIdx.x]) atomicAdd(&ctr[CTR_E_CONVEX + threadIdx.x], (u64)s_cnt[threadIdx.x]);
}

// -------------------------------------------------------------------------------------------------------------
// T5: cone angle, side bits, lowest triangle id -- combined per tile vertex in shared memory
// -------------------------------------------------------------------------------------------------------------
// unit pseudonormal of vertex v from the fixed-point sums (zero vector: no usable axis -> full sphere on both sides)
__device__ __forceinline__ void vertex_axis64(const u64 *__restrict__ vacc, size_t v, double *N) {
#pragma unroll
    for (int i = 0; i < 3; i++) N[i] = (double)(long long)vacc[3 * v + i] * (1.0 / FIXSCALE);
    const double L = sqrt(ddot(N, N));
    if (L > 1e-9) { N[0] /= L; N[1] /= L; N[2] /= L; }
    else { N[0] = 0.0; N[1] = 0.0; N[2] = 0.0; }
}

struct TileConeSmem {
    float pos[TC * 3];
    double N[TCAP * 3];
    u32 vid[TC];
    int perm[TT];
    int hi[TCAP];
    u32 lo[TCAP];
    int side[TCAP];
    int mint[TCAP];
    unsigned short lv[TC];
};

__global__ void __launch_bounds__(TB, 3) tile_cone_kernel(const float *__restrict__ soup, int F, const int *__restrict__ perm,
                                                          TileTables tt, const u64 *__restrict__ vacc,
                                                          long long *__restrict__ vcosq, int *__restrict__ vside,
                                                          int *__restrict__ vmint, long long *__restrict__ vcospos) {
    extern __shared__ __align__(16) unsigned char tile_smem[];
    TileConeSmem &S = *(TileConeSmem *)tile_smem;
    const int tid = threadIdx.x;
    const int b0 = blockIdx.x * TT;
    const int nt = min(TT, F - b0), nc = 3 * nt;
    const int nlv = tt.tnlv[blockIdx.x];
    const int nacc = min(nlv, TCAP);
    for (int j = tid; j < 9 * nt; j += TB) S.pos[j] = soup[9 * (size_t)b0 + j];
    for (int c = tid; c < nc; c += TB) S.lv[c] = tt.clv[3 * (size_t)b0 + c];
    for (int i = tid; i < nt; i += TB) S.perm[i] = perm[b0 + i];
    for (int lv = tid; lv < nlv; lv += TB) {
        const u32 v = tt.tvid[3 * (size_t)b0 + lv] & ~SHARED_BIT;
        S.vid[lv] = v;
        if (lv < TCAP) {
            vertex_axis64(vacc, v, &S.N[3 * lv]);
            S.hi[lv] = 0x7FFFFFFF; S.lo[lv] = 0xFFFFFFFFu; S.side[lv] = 0; S.mint[lv] = 0x7FFFFFFF;
        }
    }
    __syncthreads();
    // for each corner: cos of the angle between the face normal and the vertex axis (eq.9), which
    // side of the pseudonormal plane the two neighbours lie on, lowest incident triangle id
    long long key[TCPT / 3 * 3 > 0 ? 2 * 3 : 3];      // two triangles per thread, three corners each
    bool live[2] = {false, false};
#pragma unroll
    for (int r = 0; r < 2; r++) {
        const int i = tid + r * TB;
        if (i >= nt) continue;
        double n[3], p[3][3];
        if (!tri_normal64(&S.pos[9 * i], n, p)) continue;
        live[r] = true;
        const int xt = S.perm[i];                               // the caller's triangle id
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const int lv = S.lv[3 * i + k];
            double Nl[3];
            const double *N = Nl;
            if (lv < TCAP) N = &S.N[3 * lv];
            else vertex_axis64(vacc, S.vid[lv], Nl);
            const double c = ddot(n, N);
            const long long kq = (long long)floor(c * COSSCALE);
            key[3 * r + k] = kq;
            int bits = 0;
#pragma unroll
            for (int q = 1; q <= 2; q++) {
                const int kq2 = (k + q) % 3;
                const double e[3] = {p[kq2][0] - p[k][0], p[kq2][1] - p[k][1], p[kq2][2] - p[k][2]};
                const double s = ddot(e, N) / sqrt(ddot(e, e));
                bits |= (s > 1e-9) ? 1 : ((s < -1e-9) ? 2 : 4);     // above / below / on the plane
            }
            if (lv < TCAP) {
                atomicMin(&S.hi[lv], (int)(kq >> 32));
                if ((S.side[lv] & bits) != bits) atomicOr(&S.side[lv], bits);
                if (S.mint[lv] > xt) atomicMin(&S.mint[lv], xt);
            } else {
                const u32 v = S.vid[lv];
                atomicMin(&vcosq[v], kq);
                if ((vside[v] & bits) != bits) atomicOr(&vside[v], bits);
                if (vmint[v] > xt) atomicMin(&vmint[v], xt);
            }
            // ablation: the cone over the positive-pointing normals only
            if (vcospos && c > 0.0) atomicMin(&vcospos[S.vid[lv]], kq);
        }
    }
    __syncthreads();
    // the 64-bit minimum in two 32-bit steps: the high words first, then the low words of those that tie
#pragma unroll
    for (int r = 0; r < 2; r++) {
        if (!live[r]) continue;
        const int i = tid + r * TB;
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const int lv = S.lv[3 * i + k];
            if (lv < TCAP && (int)(key[3 * r + k] >> 32) == S.hi[lv]) atomicMin(&S.lo[lv], (u32)(key[3 * r + k] & 0xFFFFFFFFll));
        }
    }
    __syncthreads();
    for (int lv = tid; lv < nacc; lv += TB) {
        if (S.hi[lv] == 0x7FFFFFFF && S.lo[lv] == 0xFFFFFFFFu) continue;        // only zero-area triangles at this vertex
        const u32 v = S.vid[lv];
        const long long kq = (long long)(((u64)(u32)S.hi[lv] << 32) | (u64)S.lo[lv]);
        if (vcosq[v] > kq) atomicMin(&vcosq[v], kq);
        const int bits = S.side[lv];
        if ((vside[v] & bits) != bits) atomicOr(&vside[v], bits);
        if (vmint[v] > S.mint[lv]) atomicMin(&vmint[v], S.mint[lv]);
    }
}
