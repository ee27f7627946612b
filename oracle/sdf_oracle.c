/*
 * sdf_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 definition of what the CSC closest-point transform of
 * arXiv:1903.00353 computes: the narrow-band restriction of the exact signed
 * distance function of a closed triangle soup (eq.1; the
 * completeness argument PAPER.md:131-238 is why the CSC method reaches exactly
 * this).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  It shares no code with the CUDA path.
 *
 * Algorithm (north_star of BASELINE.json), all fp64 on the
 * fp32 inputs promoted exactly:
 *   1. x(i,j,k) = origin + (i,j,k)*h
 *   2. connectivity: vertices equal <=> bit-identical xyz (-0 == +0); every
 *      undirected edge must have exactly two triangles traversing it in
 *      opposite directions (closed, consistently oriented).
 *   3. unit face normal n = (b-a)x(c-a)/|.| (CCW from outside);
 *      corner angle alpha = atan2(|u x v|, u.v); vertex pseudonormal
 *      N_v = sum alpha_i n_i (eq.8); edge pseudonormal
 *      N_e = n_1 + n_2 ("average normal of the edge").
 *   4. for every triangle t (ascending), for every cell of its band-expanded
 *      AABB: closest point c on the triangle (seven regions: face / 3 edges /
 *      3 vertices), d = |x - c|; strict d < best keeps the lowest id on ties;
 *      sign = (N_r . (x - c) < 0) ? -1 : +1 with N_r the pseudonormal of the
 *      feature the region maps to.
 *   5. populated iff best < band (strict); dist = (float)(s*best)
 *      with -0 -> +0; elsewhere dist = +inf, tri = -1.
 *
 * Pins (tests/test_oracle_pins.py): closed-form box SDF, brute-force winding
 * numbers, dense barycentric sampling, textbook point/segment/plane special
 * cases, cube-corner pseudonormal, sphere sagitta bound, invariants.
 * Parity unpinned: full-size C4/C5 outputs beyond those invariants.
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK           0
#define ORACLE_EINVAL       1
#define ORACLE_ENOTCLOSED   2
#define ORACLE_EORIENT      3
#define ORACLE_EDEGENERATE  4
#define ORACLE_ENOMEM       5

enum { R_FACE = 0, R_EAB = 1, R_EBC = 2, R_ECA = 3, R_VA = 4, R_VB = 5, R_VC = 6 };

typedef struct oracle_mesh {
    int64_t F, V, E;
    double *pos;      /* [F][3][3] triangle corner positions (fp32 promoted)       */
    int32_t *cvid;    /* [3F] corner -> vertex id                                   */
    int32_t *ceid;    /* [3F] half-edge (corner c -> c+1) -> edge id                */
    double *fn;       /* [F][3] unit face normals                                   */
    double *vn;       /* [V][3] angle-weighted vertex pseudonormals (eq.8)          */
    double *en;       /* [E][3] edge pseudonormals n1 + n2                          */
    int32_t *eclass;  /* [E] +1 convex, -1 concave, 0 flat      */
    int32_t *vclass;  /* [V] +1 convex, -1 concave, 0 flat, 2 saddle */
    double *vcos;     /* [V] min_i n_i . N_v/|N_v|      */
} oracle_mesh;

/* ------------------------------------------------------------------ helpers */
static inline void v_sub(const double *a, const double *b, double *r) { r[0] = a[0] - b[0]; r[1] = a[1] - b[1]; r[2] = a[2] - b[2]; }
static inline double v_dot(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static inline void v_cross(const double *a, const double *b, double *r) {
    r[0] = a[1] * b[2] - a[2] * b[1]; r[1] = a[2] * b[0] - a[0] * b[2]; r[2] = a[0] * b[1] - a[1] * b[0];
}
static inline double v_norm(const double *a) { return sqrt(v_dot(a, a)); }

/* Closest point on triangle (a,b,c) to p, with the region it falls in.
 * Seven Voronoi regions of the triangle; clamped barycentric coordinates.
 * Special cases reduce to the textbook formulas of PAPER.md:392 (point-plane,
 * point-line, point-point). */
static double closest_point_triangle(const double *p, const double *a, const double *b, const double *c,
                                     double *q, int *region) {
    double ab[3], ac[3], ap[3], bp[3], cp[3], diff[3];
    v_sub(b, a, ab); v_sub(c, a, ac); v_sub(p, a, ap);
    double d1 = v_dot(ab, ap), d2 = v_dot(ac, ap);
    if (d1 <= 0.0 && d2 <= 0.0) { q[0] = a[0]; q[1] = a[1]; q[2] = a[2]; *region = R_VA; goto done; }
    v_sub(p, b, bp);
    double d3 = v_dot(ab, bp), d4 = v_dot(ac, bp);
    if (d3 >= 0.0 && d4 <= d3) { q[0] = b[0]; q[1] = b[1]; q[2] = b[2]; *region = R_VB; goto done; }
    double vc = d1 * d4 - d3 * d2;
    if (vc <= 0.0 && d1 >= 0.0 && d3 <= 0.0) {
        double v = d1 / (d1 - d3);
        for (int i = 0; i < 3; i++) q[i] = a[i] + v * ab[i];
        *region = R_EAB; goto done;
    }
    v_sub(p, c, cp);
    double d5 = v_dot(ab, cp), d6 = v_dot(ac, cp);
    if (d6 >= 0.0 && d5 <= d6) { q[0] = c[0]; q[1] = c[1]; q[2] = c[2]; *region = R_VC; goto done; }
    double vb = d5 * d2 - d1 * d6;
    if (vb <= 0.0 && d2 >= 0.0 && d6 <= 0.0) {
        double w = d2 / (d2 - d6);
        for (int i = 0; i < 3; i++) q[i] = a[i] + w * ac[i];
        *region = R_ECA; goto done;
    }
    double va = d3 * d6 - d5 * d4;
    if (va <= 0.0 && (d4 - d3) >= 0.0 && (d5 - d6) >= 0.0) {
        double w = (d4 - d3) / ((d4 - d3) + (d5 - d6));
        for (int i = 0; i < 3; i++) q[i] = b[i] + w * (c[i] - b[i]);
        *region = R_EBC; goto done;
    }
    {
        double denom = 1.0 / (va + vb + vc);
        double v = vb * denom, w = vc * denom;
        for (int i = 0; i < 3; i++) q[i] = a[i] + ab[i] * v + ac[i] * w;
        *region = R_FACE;
    }
done:
    v_sub(p, q, diff);
    return v_norm(diff);
}

/* exported: distance from p to one triangle given as 9 floats */
double oracle_point_triangle(const double *p, const float *tri9, double *closest, int *region) {
    double a[3], b[3], c[3];
    for (int i = 0; i < 3; i++) { a[i] = tri9[i]; b[i] = tri9[3 + i]; c[i] = tri9[6 + i]; }
    return closest_point_triangle(p, a, b, c, closest, region);
}

/* ------------------------------------------------------------ connectivity */
typedef struct { uint32_t x, y, z; int64_t corner; } vrec;
static int vrec_cmp(const void *pa, const void *pb) {
    const vrec *a = (const vrec *)pa, *b = (const vrec *)pb;
    if (a->x != b->x) return a->x < b->x ? -1 : 1;
    if (a->y != b->y) return a->y < b->y ? -1 : 1;
    if (a->z != b->z) return a->z < b->z ? -1 : 1;
    return a->corner < b->corner ? -1 : (a->corner > b->corner);
}
typedef struct { int32_t lo, hi; int64_t he; int32_t fwd; } erec;
static int erec_cmp(const void *pa, const void *pb) {
    const erec *a = (const erec *)pa, *b = (const erec *)pb;
    if (a->lo != b->lo) return a->lo < b->lo ? -1 : 1;
    if (a->hi != b->hi) return a->hi < b->hi ? -1 : 1;
    return a->he < b->he ? -1 : (a->he > b->he);
}
static uint32_t fbits(float f) {
    if (f == 0.0f) f = 0.0f;   /* -0 -> +0 */
    uint32_t u; memcpy(&u, &f, 4); return u;
}

void oracle_free(oracle_mesh *m) {
    if (!m) return;
    free(m->pos); free(m->cvid); free(m->ceid); free(m->fn); free(m->vn); free(m->en);
    free(m->eclass); free(m->vclass); free(m->vcos); free(m);
}

int oracle_build(const float *tri, int64_t ntri, oracle_mesh **out) {
    if (!tri || !out || ntri <= 0) return ORACLE_EINVAL;
    *out = NULL;
    int64_t F = ntri, C = 3 * ntri;
    for (int64_t i = 0; i < 9 * F; i++) if (!isfinite(tri[i])) return ORACLE_EINVAL;
    oracle_mesh *m = (oracle_mesh *)calloc(1, sizeof(oracle_mesh));
    if (!m) return ORACLE_ENOMEM;
    m->F = F;
    m->pos = (double *)malloc(sizeof(double) * 9 * F);
    m->cvid = (int32_t *)malloc(sizeof(int32_t) * C);
    m->ceid = (int32_t *)malloc(sizeof(int32_t) * C);
    m->fn = (double *)malloc(sizeof(double) * 3 * F);
    vrec *vr = (vrec *)malloc(sizeof(vrec) * C);
    erec *er = (erec *)malloc(sizeof(erec) * C);
    int status = ORACLE_OK;
    if (!m->pos || !m->cvid || !m->ceid || !m->fn || !vr || !er) { status = ORACLE_ENOMEM; goto fail; }
    for (int64_t i = 0; i < 9 * F; i++) m->pos[i] = (tri[i] == 0.0f) ? 0.0 : (double)tri[i];

    /* weld: identical <=> bit-identical fp32 triple */
    for (int64_t c = 0; c < C; c++) {
        vr[c].x = fbits(tri[3 * c]); vr[c].y = fbits(tri[3 * c + 1]); vr[c].z = fbits(tri[3 * c + 2]);
        vr[c].corner = c;
    }
    qsort(vr, (size_t)C, sizeof(vrec), vrec_cmp);
    int64_t V = 0;
    for (int64_t i = 0; i < C; i++) {
        if (i > 0 && (vr[i].x != vr[i - 1].x || vr[i].y != vr[i - 1].y || vr[i].z != vr[i - 1].z)) V++;
        m->cvid[vr[i].corner] = (int32_t)V;
    }
    V++;
    m->V = V;

    /* degenerate: repeated vertex or zero area */
    for (int64_t t = 0; t < F; t++) {
        int32_t *v = m->cvid + 3 * t;
        if (v[0] == v[1] || v[1] == v[2] || v[2] == v[0]) { status = ORACLE_EDEGENERATE; goto fail; }
        const double *a = m->pos + 9 * t, *b = a + 3, *c = a + 6;
        double ab[3], ac[3], n[3];
        v_sub(b, a, ab); v_sub(c, a, ac); v_cross(ab, ac, n);
        double L = v_norm(n);
        if (!(L > 0.0)) { status = ORACLE_EDEGENERATE; goto fail; }
        m->fn[3 * t] = n[0] / L; m->fn[3 * t + 1] = n[1] / L; m->fn[3 * t + 2] = n[2] / L;
    }

    /* edges: half-edge c goes corner c -> corner (c+1)%3 of its triangle */
    if (C % 2) { status = ORACLE_ENOTCLOSED; goto fail; }
    for (int64_t t = 0; t < F; t++)
        for (int c = 0; c < 3; c++) {
            int32_t u = m->cvid[3 * t + c], w = m->cvid[3 * t + (c + 1) % 3];
            erec *e = er + 3 * t + c;
            e->lo = u < w ? u : w; e->hi = u < w ? w : u; e->he = 3 * t + c; e->fwd = (u < w);
        }
    qsort(er, (size_t)C, sizeof(erec), erec_cmp);
    for (int64_t i = 0; i < C; ) {
        int64_t j = i;
        while (j < C && er[j].lo == er[i].lo && er[j].hi == er[i].hi) j++;
        if (j - i != 2) { status = ORACLE_ENOTCLOSED; goto fail; }
        i = j;
    }
    for (int64_t i = 0; i < C; i += 2)
        if (er[i].fwd == er[i + 1].fwd) { status = ORACLE_EORIENT; goto fail; }
    int64_t E = C / 2;
    m->E = E;
    m->vn = (double *)calloc((size_t)(3 * V), sizeof(double));
    m->en = (double *)calloc((size_t)(3 * E), sizeof(double));
    m->eclass = (int32_t *)calloc((size_t)E, sizeof(int32_t));
    m->vclass = (int32_t *)calloc((size_t)V, sizeof(int32_t));
    m->vcos = (double *)malloc(sizeof(double) * V);
    if (!m->vn || !m->en || !m->eclass || !m->vclass || !m->vcos) { status = ORACLE_ENOMEM; goto fail; }

    for (int64_t e = 0; e < E; e++) {
        int64_t h1 = er[2 * e].he, h2 = er[2 * e + 1].he;
        m->ceid[h1] = (int32_t)e; m->ceid[h2] = (int32_t)e;
        const double *n1 = m->fn + 3 * (h1 / 3), *n2 = m->fn + 3 * (h2 / 3);
        for (int i = 0; i < 3; i++) m->en[3 * e + i] = n1[i] + n2[i];
        /* discriminant d = (ab x n1) . n2 with ab the direction of the half-edge in
         * the triangle that owns n1 */
        const double *a = m->pos + 3 * h1, *b = m->pos + 3 * (3 * (h1 / 3) + (h1 % 3 + 1) % 3);
        double ab[3], x[3];
        v_sub(b, a, ab); v_cross(ab, n1, x);
        double d = v_dot(x, n2) / v_norm(ab);
        m->eclass[e] = d > 1e-12 ? 1 : (d < -1e-12 ? -1 : 0);
    }

    /* vertex pseudonormals, eq.8: N_v = sum alpha_i n_i */
    for (int64_t t = 0; t < F; t++)
        for (int c = 0; c < 3; c++) {
            const double *p0 = m->pos + 9 * t + 3 * c, *p1 = m->pos + 9 * t + 3 * ((c + 1) % 3),
                         *p2 = m->pos + 9 * t + 3 * ((c + 2) % 3);
            double u[3], w[3], x[3];
            v_sub(p1, p0, u); v_sub(p2, p0, w); v_cross(u, w, x);
            double alpha = atan2(v_norm(x), v_dot(u, w));
            int32_t v = m->cvid[3 * t + c];
            for (int i = 0; i < 3; i++) m->vn[3 * v + i] += alpha * m->fn[3 * t + i];
        }
    /* vertex classes: sign of (v_n - v).N_v over all neighbours (
     * reading #2 of SURVEY.md 8(c): convex <=> all neighbours below the plane) */
    {
        int32_t *npos = (int32_t *)calloc((size_t)V, sizeof(int32_t));
        int32_t *nneg = (int32_t *)calloc((size_t)V, sizeof(int32_t));
        if (!npos || !nneg) { free(npos); free(nneg); status = ORACLE_ENOMEM; goto fail; }
        for (int64_t v = 0; v < V; v++) m->vcos[v] = 2.0;
        for (int64_t t = 0; t < F; t++)
            for (int c = 0; c < 3; c++) {
                int32_t v = m->cvid[3 * t + c];
                const double *N = m->vn + 3 * v;
                double L = v_norm(N);
                const double *p0 = m->pos + 9 * t + 3 * c;
                double cs = v_dot(m->fn + 3 * t, N) / L;
                if (cs < m->vcos[v]) m->vcos[v] = cs;
                for (int k = 1; k <= 2; k++) {
                    const double *pk = m->pos + 9 * t + 3 * ((c + k) % 3);
                    double e[3]; v_sub(pk, p0, e);
                    double d = v_dot(e, N) / (L * v_norm(e));
                    if (d > 1e-12) npos[v]++; else if (d < -1e-12) nneg[v]++;
                }
            }
        for (int64_t v = 0; v < V; v++)
            m->vclass[v] = (npos[v] && nneg[v]) ? 2 : (nneg[v] ? 1 : (npos[v] ? -1 : 0));
        free(npos); free(nneg);
    }
    free(vr); free(er);
    *out = m;
    return ORACLE_OK;
fail:
    free(vr); free(er); oracle_free(m);
    return status;
}

/* out[0..9] = F, V, E, convex_e, concave_e, flat_e, convex_v, concave_v, flat_v, saddle_v */
void oracle_counts(const oracle_mesh *m, int64_t *out) {
    memset(out, 0, sizeof(int64_t) * 10);
    out[0] = m->F; out[1] = m->V; out[2] = m->E;
    for (int64_t e = 0; e < m->E; e++) out[m->eclass[e] > 0 ? 3 : (m->eclass[e] < 0 ? 4 : 5)]++;
    for (int64_t v = 0; v < m->V; v++)
        out[m->vclass[v] == 1 ? 6 : (m->vclass[v] == -1 ? 7 : (m->vclass[v] == 0 ? 8 : 9))]++;
}
void oracle_get_corner_vid(const oracle_mesh *m, int32_t *out) { memcpy(out, m->cvid, sizeof(int32_t) * 3 * m->F); }
void oracle_get_corner_eid(const oracle_mesh *m, int32_t *out) { memcpy(out, m->ceid, sizeof(int32_t) * 3 * m->F); }
void oracle_get_vertex_normals(const oracle_mesh *m, double *out) { memcpy(out, m->vn, sizeof(double) * 3 * m->V); }
void oracle_get_edge_normals(const oracle_mesh *m, double *out) { memcpy(out, m->en, sizeof(double) * 3 * m->E); }
void oracle_get_face_normals(const oracle_mesh *m, double *out) { memcpy(out, m->fn, sizeof(double) * 3 * m->F); }
void oracle_get_classes(const oracle_mesh *m, int32_t *eclass, int32_t *vclass, double *vcos) {
    if (eclass) memcpy(eclass, m->eclass, sizeof(int32_t) * m->E);
    if (vclass) memcpy(vclass, m->vclass, sizeof(int32_t) * m->V);
    if (vcos) memcpy(vcos, m->vcos, sizeof(double) * m->V);
}

/* pseudonormal of the feature that region r of triangle t maps to */
static const double *region_normal(const oracle_mesh *m, int64_t t, int r) {
    switch (r) {
    case R_FACE: return m->fn + 3 * t;
    case R_EAB:  return m->en + 3 * (int64_t)m->ceid[3 * t + 0];
    case R_EBC:  return m->en + 3 * (int64_t)m->ceid[3 * t + 1];
    case R_ECA:  return m->en + 3 * (int64_t)m->ceid[3 * t + 2];
    case R_VA:   return m->vn + 3 * (int64_t)m->cvid[3 * t + 0];
    case R_VB:   return m->vn + 3 * (int64_t)m->cvid[3 * t + 1];
    default:     return m->vn + 3 * (int64_t)m->cvid[3 * t + 2];
    }
}

/* ---------------------------------------------------------------- the SDF */
typedef struct {
    const oracle_mesh *m; const double *origin; double h, band; int nx, ny, nz;
    int k_lo, k_hi;           /* slab owned by this thread: k in [k_lo, k_hi) */
    double *best; int8_t *sgn; int32_t *id;
} slab_job;

static void *slab_run(void *arg) {
    slab_job *J = (slab_job *)arg;
    const oracle_mesh *m = J->m;
    const double h = J->h, band = J->band, *o = J->origin;
    const int dims[3] = { J->nx, J->ny, J->nz };
    for (int64_t t = 0; t < m->F; t++) {
        const double *a = m->pos + 9 * t, *b = a + 3, *c = a + 6;
        int lo[3], hi[3], empty = 0;
        for (int ax = 0; ax < 3; ax++) {
            double mn = fmin(a[ax], fmin(b[ax], c[ax])), mx = fmax(a[ax], fmax(b[ax], c[ax]));
            double l = ceil((mn - band - o[ax]) / h) - 1.0, u = floor((mx + band - o[ax]) / h) + 1.0;
            if (l < 0.0) l = 0.0;
            if (u > dims[ax] - 1) u = dims[ax] - 1;
            if (l > u) { empty = 1; break; }
            lo[ax] = (int)l; hi[ax] = (int)u;
        }
        if (empty) continue;
        if (lo[2] < J->k_lo) lo[2] = J->k_lo;
        if (hi[2] > J->k_hi - 1) hi[2] = J->k_hi - 1;
        for (int k = lo[2]; k <= hi[2]; k++)
            for (int j = lo[1]; j <= hi[1]; j++)
                for (int i = lo[0]; i <= hi[0]; i++) {
                    double x[3] = { o[0] + i * h, o[1] + j * h, o[2] + k * h }, q[3], diff[3];
                    int r;
                    double d = closest_point_triangle(x, a, b, c, q, &r);
                    int64_t cell = ((int64_t)k * J->ny + j) * J->nx + i;
                    if (d < J->best[cell]) {
                        J->best[cell] = d;
                        J->id[cell] = (int32_t)t;
                        v_sub(x, q, diff);
                        J->sgn[cell] = (v_dot(region_normal(m, t, r), diff) < 0.0) ? -1 : 1;
                    }
                }
    }
    return NULL;
}

/* Narrow-band signed distance grid.  dist/tri_out: caller-owned, nx*ny*nz each. */
int oracle_sdf(const oracle_mesh *m, const double *origin, double h, int nx, int ny, int nz, double band,
               float *dist, int32_t *tri_out, int nthreads) {
    if (!m || !origin || !dist || !tri_out || !(h > 0.0) || !(band > 0.0) || nx <= 0 || ny <= 0 || nz <= 0)
        return ORACLE_EINVAL;
    int64_t N = (int64_t)nx * ny * nz;
    double *best = (double *)malloc(sizeof(double) * N);
    int8_t *sgn = (int8_t *)malloc((size_t)N);
    if (!best || !sgn) { free(best); free(sgn); return ORACLE_ENOMEM; }
    for (int64_t i = 0; i < N; i++) { best[i] = INFINITY; sgn[i] = 1; tri_out[i] = -1; }
    if (nthreads < 1) nthreads = 1;
    if (nthreads > nz) nthreads = nz;
    pthread_t *th = (pthread_t *)malloc(sizeof(pthread_t) * nthreads);
    slab_job *jobs = (slab_job *)malloc(sizeof(slab_job) * nthreads);
    for (int i = 0; i < nthreads; i++) {
        slab_job J = { m, origin, h, band, nx, ny, nz, (int)((int64_t)nz * i / nthreads),
                       (int)((int64_t)nz * (i + 1) / nthreads), best, sgn, tri_out };
        jobs[i] = J;
        if (nthreads > 1) pthread_create(&th[i], NULL, slab_run, &jobs[i]);
    }
    if (nthreads == 1) slab_run(&jobs[0]);
    else for (int i = 0; i < nthreads; i++) pthread_join(th[i], NULL);
    for (int64_t i = 0; i < N; i++) {
        if (best[i] < band) {
            float f = (float)(sgn[i] * best[i]);
            dist[i] = (f == 0.0f) ? 0.0f : f;
        } else { dist[i] = INFINITY; tri_out[i] = -1; }
    }
    free(best); free(sgn); free(th); free(jobs);
    return ORACLE_OK;
}

/* ------------------------------------------- brute-force point queries (eq.1) */
typedef struct { const oracle_mesh *m; const double *pts; int64_t lo, hi; double *d; int32_t *id; } query_job;
static void *query_run(void *arg) {
    query_job *J = (query_job *)arg;
    const oracle_mesh *m = J->m;
    for (int64_t p = J->lo; p < J->hi; p++) {
        const double *x = J->pts + 3 * p;
        double best = INFINITY, q[3], diff[3]; int32_t id = -1; int sg = 1;
        for (int64_t t = 0; t < m->F; t++) {
            const double *a = m->pos + 9 * t; int r;
            double d = closest_point_triangle(x, a, a + 3, a + 6, q, &r);
            if (d < best) {
                best = d; id = (int32_t)t;
                v_sub(x, q, diff);
                sg = (v_dot(region_normal(m, t, r), diff) < 0.0) ? -1 : 1;
            }
        }
        J->d[p] = sg * best; J->id[p] = id;
    }
    return NULL;
}
/* signed distance (fp64, no band) and closest triangle for arbitrary points */
int oracle_query(const oracle_mesh *m, const double *pts, int64_t npts, double *d_out, int32_t *id_out, int nthreads) {
    if (!m || !pts || !d_out || !id_out || npts < 0) return ORACLE_EINVAL;
    if (nthreads < 1) nthreads = 1;
    if (nthreads > npts) nthreads = npts > 0 ? (int)npts : 1;
    pthread_t *th = (pthread_t *)malloc(sizeof(pthread_t) * nthreads);
    query_job *jobs = (query_job *)malloc(sizeof(query_job) * nthreads);
    for (int i = 0; i < nthreads; i++) {
        query_job J = { m, pts, npts * i / nthreads, npts * (i + 1) / nthreads, d_out, id_out };
        jobs[i] = J;
        pthread_create(&th[i], NULL, query_run, &jobs[i]);
    }
    for (int i = 0; i < nthreads; i++) pthread_join(th[i], NULL);
    free(th); free(jobs);
    return ORACLE_OK;
}

/* unsigned fp64 distance from each point to one named triangle of the mesh
 * (used by the comparison harness for the closest-id tolerance clause) */
int oracle_dist_to_triangles(const oracle_mesh *m, const double *pts, const int32_t *tri_ids, int64_t npts, double *d_out) {
    if (!m || !pts || !tri_ids || !d_out) return ORACLE_EINVAL;
    for (int64_t p = 0; p < npts; p++) {
        int64_t t = tri_ids[p];
        if (t < 0 || t >= m->F) { d_out[p] = INFINITY; continue; }
        const double *a = m->pos + 9 * t; double q[3]; int r;
        d_out[p] = closest_point_triangle(pts + 3 * p, a, a + 3, a + 6, q, &r);
    }
    return ORACLE_OK;
}

/*
 * oracle_fill_interior -- SURVEY.md 8(f) NEXT-1.  PAPER.md:493 (sec.11.3): the narrow band
 * "lead[s] to a secondary zero crossing between the negative limit of the SDF and the interior
 * of the surface beyond the maximum distance.  This can be easily fixed by sweeping along each of
 * the coordinate axes and filling in unset values in the interior of the geometry."
 *
 * Written out as stated: for the axes x, y, z in turn, every grid line is walked forward and then
 * backward, in place.  Walking a line keeps the sign of the last set cell seen (nothing before
 * the first); an unset cell (+inf) met while that sign is negative lies in the interior and is set
 * to -band, the negative limit of the narrow-band SDF.  Cells set by an earlier walk count as set
 * for the later ones.  Exterior cells stay +inf.
 */
static void fill_line(float *d, int64_t n, int64_t stride, float fillv) {
    for (int dir = 0; dir < 2; dir++) {
        int state = 0;
        for (int64_t q = 0; q < n; q++) {
            float *c = d + (dir ? (n - 1 - q) : q) * stride;
            if (isfinite(*c)) state = (*c < 0.0f) ? -1 : 1;
            else if (state < 0) *c = fillv;
        }
    }
}

int oracle_fill_interior(float *dist, int nx, int ny, int nz, float band) {
    if (!dist || nx <= 0 || ny <= 0 || nz <= 0 || !(band > 0.0f)) return ORACLE_EINVAL;
    const float fillv = -band;
    const int64_t sx = 1, sy = nx, sz = (int64_t)nx * ny;
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++) fill_line(dist + k * sz + j * sy, nx, sx, fillv);
    for (int k = 0; k < nz; k++)
        for (int i = 0; i < nx; i++) fill_line(dist + k * sz + i * sx, ny, sy, fillv);
    for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) fill_line(dist + j * sy + i * sx, nz, sz, fillv);
    return ORACLE_OK;
}

/*
 * oracle_closest_points -- SURVEY.md 8(f) NEXT-2: the closest point transform proper
 * ("the closest point transform ... computes the closest point on the surface" beside
 * the distance).  Plain definition: for every cell with a closest-triangle id t >= 0 the point of
 * triangle t nearest to the cell centre x = origin + (i,j,k)*h (same seven-region routine as the
 * distance, fp64); +inf in the three components elsewhere.
 */
int oracle_closest_points(const oracle_mesh *m, const double *origin, double h, int nx, int ny, int nz,
                          const int32_t *tri, float *cp_out) {
    if (!m || !origin || !tri || !cp_out || nx <= 0 || ny <= 0 || nz <= 0) return ORACLE_EINVAL;
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                const int64_t c = ((int64_t)k * ny + j) * nx + i;
                float *o = cp_out + 3 * c;
                const int32_t t = tri[c];
                if (t < 0 || t >= m->F) { o[0] = o[1] = o[2] = INFINITY; continue; }
                const double p[3] = {origin[0] + i * h, origin[1] + j * h, origin[2] + k * h};
                const double *T = m->pos + 9 * (int64_t)t;
                double q[3];
                int region;
                closest_point_triangle(p, T, T + 3, T + 6, q, &region);
                o[0] = (float)q[0]; o[1] = (float)q[1]; o[2] = (float)q[2];
            }
    return ORACLE_OK;
}
