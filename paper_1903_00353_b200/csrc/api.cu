// api.cu -- the C ABI of include/sdf.h: argument checks, handle lifetime, allocator plumbing.
#include "common.cuh"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <new>

int g_last_cuda_error = 0;
int g_timing = 0;
long long g_launch_count = 0;

void stage_mark(sdf_mesh *m, int stage, int which, cudaStream_t st) {
    if (!g_timing || (g_timing == 2 && stage != SDF_T_FILL)) return;
    if (!m->ev[stage][which] && cudaEventCreate(&m->ev[stage][which]) != cudaSuccess) {
        m->ev[stage][which] = nullptr;
        (void)cudaGetLastError();
        return;
    }
    cudaEventRecord(m->ev[stage][which], st);
    if (which == 1) m->ev_set[stage] = true;
}

#include <mutex>
#include <vector>
static std::mutex g_ev_mutex;
static std::vector<cudaEvent_t> g_ev_pool[64];      // per device: idle events (cudaEventDisableTiming)
int ev_get(sdf_mesh *m, cudaEvent_t *e) {
    if (*e) return SDF_OK;
    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (!m->ev_dev1) m->ev_dev1 = dev + 1;
    if (m->ev_dev1 == dev + 1 && dev >= 0 && dev < 64) {
        std::lock_guard<std::mutex> lk(g_ev_mutex);
        if (!g_ev_pool[dev].empty()) { *e = g_ev_pool[dev].back(); g_ev_pool[dev].pop_back(); return SDF_OK; }
    }
    CK(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
    return SDF_OK;
}
void ev_put(sdf_mesh *m, cudaEvent_t *e) {
    if (!*e) return;
    int dev = -1;
    // back to the pool of the device it was taken on (a handle used on another device keeps its events out of the pools)
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64 && m->ev_dev1 == dev + 1) {
        std::lock_guard<std::mutex> lk(g_ev_mutex);
        if (g_ev_pool[dev].size() < 256) { g_ev_pool[dev].push_back(*e); *e = nullptr; return; }
    }
    cudaEventDestroy(*e);
    *e = nullptr;
}

int dev_alloc(const sdf_allocator *a, void **p, size_t bytes, cudaStream_t st) {
    *p = nullptr;
    if (bytes == 0) bytes = 16;
    if (a && a->alloc) {
        *p = a->alloc(bytes, (void *)st, a->user);
        return *p ? SDF_OK : SDF_ENOMEM;
    }
    cudaError_t e = cudaMallocAsync(p, bytes, st);
    if (e != cudaSuccess) {
        g_last_cuda_error = (int)e;
        (void)cudaGetLastError();
        *p = nullptr;
        return e == cudaErrorMemoryAllocation ? SDF_ENOMEM : SDF_ECUDA;
    }
    return SDF_OK;
}

void dev_free(const sdf_allocator *a, void *p, cudaStream_t st) {
    if (!p) return;
    if (a && a->alloc) { a->free(p, a->user); return; }
    cudaFreeAsync(p, st);
}

static int have_device() {
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n <= 0) {
        g_last_cuda_error = (int)(e != cudaSuccess ? e : cudaErrorNoDevice);
        (void)cudaGetLastError();
        return 0;
    }
    return 1;
}

extern "C" {

int sdf_version(void) { return 100; }
int64_t sdf_launch_count(void) { return (int64_t)g_launch_count; }
int sdf_enable_timing(int on) { g_timing = on == 2 ? 2 : (on ? 1 : 0); return SDF_OK; }

int sdf_get_timings(sdf_mesh *m, float *ms, int n) {
    if (!m || !ms || n != SDF_T_COUNT) return SDF_EINVAL;
    CK(cudaStreamSynchronize(m->last_stream));
    for (int i = 0; i < SDF_T_COUNT; i++) {
        ms[i] = 0.0f;
        if (m->ev_set[i] && m->ev[i][0] && m->ev[i][1]) CK(cudaEventElapsedTime(&ms[i], m->ev[i][0], m->ev[i][1]));
    }
    return SDF_OK;
}
int sdf_last_cuda_error(void) { return g_last_cuda_error; }

const char *sdf_strerror(int s) {
    switch (s) {
    case SDF_OK: return "ok";
    case SDF_EINVAL: return "invalid argument or non-finite input";
    case SDF_ENOTCLOSED: return "surface not closed: an edge without exactly two triangles";
    case SDF_EORIENT: return "inconsistent orientation: an edge traversed twice in the same direction";
    case SDF_EDEGENERATE: return "degenerate triangle (zero area or repeated vertex)";
    case SDF_ENOMEM: return "out of memory";
    case SDF_ECUDA: return "CUDA error or no CUDA device";
    case SDF_EIO: return "file cannot be opened, read or written, or is not a valid STL file";
    case SDF_ETOOBIG: return "grid too large for the static scratch of sdf_fill_interior_static (8 MiB: ny * nz * ceil(nx / 1024) <= 2^20)";
    default: return "unknown status";
    }
}

void sdf_destroy(sdf_mesh *m) {
    if (!m) return;
    cudaStream_t st = m->last_stream;
    cudaStreamSynchronize(st);
    if (m->side) cudaStreamSynchronize(m->side);      // shared, process-lifetime stream: not destroyed here
    ev_put(m, &m->ev_fork);
    ev_put(m, &m->ev_join);
    ev_put(m, &m->ev_bjoin);
    ev_put(m, &m->ev_ffork);
    ev_put(m, &m->ev_fjoin);
    void *ptrs[] = {m->slab_f, m->slab_ws, m->scratch, m->cp_state};      // (fill_state, hoist_g_dev: views into slab_f)
    for (size_t i = 0; i < sizeof(ptrs) / sizeof(ptrs[0]); i++) dev_free(&m->alloc, ptrs[i], st);
    for (int i = 0; i < SDF_T_COUNT; i++)
        for (int w = 0; w < 2; w++)
            if (m->ev[i][w]) cudaEventDestroy(m->ev[i][w]);
    m->~sdf_mesh();
    free(m);
}

static int new_mesh(int64_t ntri, const sdf_allocator *a, void *stream, sdf_mesh **out) {
    void *mem = calloc(1, sizeof(sdf_mesh));
    if (!mem) return SDF_ENOMEM;
    sdf_mesh *m = new (mem) sdf_mesh;
    memset(m, 0, sizeof(*m));
    if (a) m->alloc = *a;
    m->F = ntri;
    m->last_stream = (cudaStream_t)stream;
    *out = m;
    return SDF_OK;
}

int sdf_create(const float *tri_xyz, int64_t ntri, int on_device, const sdf_allocator *a, void *stream,
               sdf_mesh **out) {
    if (out) *out = nullptr;
    if (!tri_xyz || !out || ntri <= 0 || ntri > ((int64_t)1 << 29)) return SDF_EINVAL;
    if (a && (!a->alloc || !a->free)) return SDF_EINVAL;
    if (!have_device()) return SDF_ECUDA;
    sdf_mesh *m = nullptr;
    CKS(new_mesh(ntri, a, stream, &m));
    int s = build_features(m, tri_xyz, on_device, (cudaStream_t)stream);
    if (s != SDF_OK) {
        sdf_destroy(m);
        return s;
    }
    *out = m;
    return SDF_OK;
}

static int make_grid(const float origin[3], float h, int nx, int ny, int nz, float band, const float *dist,
                     const int32_t *tri, GridParams *g) {
    if (!origin || !(h > 0.0f) || !(band > 0.0f) || !isfinite(h) || !isfinite(band)) return SDF_EINVAL;
    if (nx <= 0 || ny <= 0 || nz <= 0 || nx > 32767 || ny > 32767 || nz > 32767) return SDF_EINVAL;
    // features flatter than 1e-6 rad are dropped (reading #5): the sliver they would cover,
    // 1e-6 * band thick, must stay inside the eps = 1e-3 * h inflation of their neighbours
    if (band > 250.0f * h) return SDF_EINVAL;
    if (!isfinite(origin[0]) || !isfinite(origin[1]) || !isfinite(origin[2])) return SDF_EINVAL;
    memset(g, 0, sizeof(*g));
    g->ox = origin[0]; g->oy = origin[1]; g->oz = origin[2]; g->h = h; g->inv_h = 1.0f / h;
    g->dox = origin[0]; g->doy = origin[1]; g->doz = origin[2]; g->dh = h;
    g->nx = nx; g->ny = ny; g->nz = nz;
    g->nbx = (nx + BRICK - 1) / BRICK; g->nby = (ny + BRICK - 1) / BRICK; g->nbz = (nz + BRICK - 1) / BRICK;
    g->band = band; g->dband = band;
    // eps: tolerance of every inclusion test, the upper value of PAPER.md:386 (1e-3 dx)
    g->eps = 1e-3f * h;
    // guard: bound on the fp32 error of an evaluated distance; cells with |d - band| < guard
    // are decided in fp64 by the emit pass
    float maxabs = 0.0f;
    const int n[3] = {nx, ny, nz};
    for (int i = 0; i < 3; i++) {
        float lo = fabsf(origin[i]), hi = fabsf(origin[i] + (n[i] - 1) * h);
        maxabs = fmaxf(maxabs, fmaxf(lo, hi));
    }
    g->guard = 1e-3f * h + 1e-6f * maxabs;
    g->tiny_abs = 2.5e-7f * maxabs;
    g->rb = band + g->guard + g->eps;
    const char *dbg = getenv("SDF_AABB_MODE");
    g->aabb_mode = (dbg && dbg[0] == '1') ? 1 : 0;
    // harness self-test: leave an extrusion class out and watch parity break
    const char *dis = getenv("SDF_DISABLE");
    g->disable = !dis ? 0 : ((strstr(dis, "faces") ? 1 : 0) | (strstr(dis, "wedges") ? 2 : 0) | (strstr(dis, "cones") ? 4 : 0));
    const char *pf = getenv("SDF_FILL_MODE");
    g->fill_mode = (pf && pf[0] >= '0' && pf[0] <= '4') ? pf[0] - '0' : 4;
    const char *fd = getenv("SDF_FILL_DEPTH"), *fi = getenv("SDF_FILL_ISSUERS");
    const char *pc = getenv("SDF_CPT_PLAIN");
    g->plain_cpt = (pc && pc[0] == '1') ? 1 : 0;
    const char *sc = getenv("SDF_SCHEDULER");
    g->serial_loop = (sc && !strcmp(sc, "serial")) ? 1 : 0;
    g->cdp = (sc && !strncmp(sc, "dynamic", 7) && (sc[7] == 0 || sc[7] == ':')) ? 1 : 0;
    g->cdp_serial_below = (g->cdp && sc[7] == ':') ? atoi(sc + 8) : 0;
    if (g->cdp_serial_below < 0) g->cdp_serial_below = 0;
    const char *fp = getenv("SDF_FILL_PRIO");
    g->fill_prio = fp ? (fp[0] == '1') : 1;
    const char *fl = getenv("SDF_FILL_CTAS");
    g->fill_ctas = fl ? atoi(fl) : 32;
    if (g->fill_ctas < 1 || g->fill_ctas > 64) g->fill_ctas = 32;
    // one issuing lane per SM, 8 KiB bulk copies, three pairs in flight: the fewer bulk stores are queued in L2 the less
    // the kernels beside the fill are held up (4 lanes x 9 pairs of 4 KiB: C4 3.27 -> 3.20 ms, C5 4.22 -> 4.12; alone the
    // fill runs at 7.3 TB/s either way; profiles/r2_ablations.md)
    g->fill_depth = fd ? atoi(fd) : 2;
    g->fill_issuers = fi ? atoi(fi) : 1;
    if (g->fill_issuers < 1 || g->fill_issuers > 4) g->fill_issuers = 1;
    const char *rcl = getenv("SDF_ROW_CLIP");
    g->row_clip = rcl ? atoi(rcl) : 2;              // (8, the first setting: C4 3.15 against 3.13 ms, C3 0.379 / 0.370, C2 0.248 / 0.241)
    if (g->row_clip < 0 || g->row_clip > 1024) g->row_clip = 2;
    const char *ec = getenv("SDF_EVAL_CHUNK");
    g->eval_chunk = ec ? atoi(ec) : 256;            // SDF_EVAL_CHUNK=0: faces, then wedges, then cones (C5: 3.99 against 3.95 ms)
    if (g->eval_chunk < 0 || g->eval_chunk > (1 << 20)) g->eval_chunk = 256;
    const char *sh = getenv("SDF_SCRATCH_HINT");
    g->scratch_hint = (sh && sh[0] == '0') ? 0 : 1;
    const char *fck = getenv("SDF_FILL_CHUNK_LOG2");
    g->fill_chunk_log2 = fck ? atoi(fck) : 13;
    if (g->fill_chunk_log2 < 11 || g->fill_chunk_log2 > 14) g->fill_chunk_log2 = 13;
    const char *fsh = getenv("SDF_FILL_SM_SHARE");
    g->fill_sm_share = fsh ? atoi(fsh) : 8;
    if (g->fill_sm_share < 1 || g->fill_sm_share > 8) g->fill_sm_share = 8;
    g->vec4 = (nx % 4 == 0) && (((uintptr_t)dist & 15) == 0) && (((uintptr_t)tri & 15) == 0);
    return SDF_OK;
}

int sdf_compute(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz, float band, float *dist_out,
                int32_t *tri_out, void *stream) {
    if (!m || !dist_out || !tri_out) return SDF_EINVAL;
    GridParams g;
    CKS(make_grid(origin, h, nx, ny, nz, band, dist_out, tri_out, &g));
    int s = run_compute(m, g, dist_out, tri_out, (cudaStream_t)stream);
    if (s != SDF_OK && m->side) cudaStreamSynchronize(m->side);   // never leave the fill in flight on failure
    return s;
}

int sdf_transform(const float *tri_xyz, int64_t ntri, int on_device, const sdf_allocator *a, const float origin[3],
                  float h, int nx, int ny, int nz, float band, float *dist_out, int32_t *tri_out, void *stream,
                  sdf_mesh **out) {
    if (out) *out = nullptr;
    if (!tri_xyz || !out || ntri <= 0 || ntri > ((int64_t)1 << 29)) return SDF_EINVAL;
    if (a && (!a->alloc || !a->free)) return SDF_EINVAL;
    if (!dist_out || !tri_out) return SDF_EINVAL;
    GridParams g;
    CKS(make_grid(origin, h, nx, ny, nz, band, dist_out, tri_out, &g));
    if (!have_device()) return SDF_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;
    sdf_mesh *m = nullptr;
    CKS(new_mesh(ntri, a, stream, &m));
    // the sentinel fill (A8a) needs only the output pointers: build_features starts it at the stage boundary
    // SDF_PREFILL_AT (1 before A0, 2 before the edge table, 3 before edge pairing, 4 = default: behind the last feature
    // kernel, i.e. under the host crossing; 5: run_compute forks it after the crossing, as the two calls do).
    // Measured: the feature kernels are bound by the same memory pipe as the fill -- beside it each is
    // stretched by what the fill moves meanwhile, whatever the fill's rate -- so 1..3 lose; only the instruction-bound
    // evaluate kernels hide it.
    const bool pre = g.fill_mode < 2 || g.fill_mode == 4;
    const char *pa = getenv("SDF_PREFILL_AT");
    m->pre_at = (pa && pa[0] >= '1' && pa[0] <= '5') ? pa[0] - '0' : 4;
    m->pre_g = pre ? &g : nullptr;
    m->pre_dist = dist_out;
    m->pre_tri = tri_out;
    // A6a (brick marks + scan, 0.2 ms at C4) needs the soup, the face normals and the grid, not the edge table:
    // build_features runs it on the vertex stream beside the edge stage, and its total comes back with the
    // validation flags -- one host crossing fewer (SDF_HOIST_BRICKS=0: leave it to run_compute)
    const char *hb = getenv("SDF_HOIST_BRICKS");
    m->hoist_g = (hb && hb[0] == '0') ? nullptr : &g;
    int s = build_features(m, tri_xyz, on_device, st);
    const bool started = pre && !m->pre_g;
    m->pre_g = nullptr;
    m->hoist_g = nullptr;
    if (s == SDF_OK) s = run_compute(m, g, dist_out, tri_out, st, started);
    if (s != SDF_OK) {
        if (m->side) cudaStreamSynchronize(m->side);   // never leave the fill in flight on failure
        sdf_destroy(m);
        return s;
    }
    *out = m;
    return SDF_OK;
}

int sdf_zslab(int nz, int part, int parts, int *k0, int *nk) {
    if (!k0 || !nk || nz < 1 || parts < 1 || part < 0 || part >= parts) return SDF_EINVAL;
    const int64_t nb = ((int64_t)nz + BRICK - 1) / BRICK;          // slabs are whole bricks high
    int64_t a = nb * part / parts * BRICK, b = nb * ((int64_t)part + 1) / parts * BRICK;
    if (a > nz) a = nz;
    if (b > nz) b = nz;
    *k0 = (int)a;
    *nk = (int)(b - a);
    return SDF_OK;
}

int sdf_compute_zslab(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz, float band, int part,
                      int parts, float *dist_out, int32_t *tri_out, void *stream, int *k0_out, int *nk_out) {
    if (!m || !origin) return SDF_EINVAL;
    int k0 = 0, nk = 0;
    CKS(sdf_zslab(nz, part, parts, &k0, &nk));
    if (k0_out) *k0_out = k0;
    if (nk_out) *nk_out = nk;
    if (nk == 0) return SDF_OK;
    const float o[3] = {origin[0], origin[1], (float)((double)origin[2] + (double)k0 * (double)h)};
    return sdf_compute(m, o, h, nx, ny, nk, band, dist_out, tri_out, stream);
}

int sdf_closest_points(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz, const int32_t *tri_in,
                       float *cp_out, void *stream) {
    if (!m || !tri_in || !cp_out) return SDF_EINVAL;
    GridParams g;
    CKS(make_grid(origin, h, nx, ny, nz, h, nullptr, nullptr, &g));      // the band plays no part here
    return run_closest_points(m, g, tri_in, cp_out, (cudaStream_t)stream);
}

int sdf_compute_host(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz, float band,
                     float *dist_out_host, int32_t *tri_out_host, void *stream) {
    if (!m || !dist_out_host || !tri_out_host) return SDF_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    GridParams g;
    CKS(make_grid(origin, h, nx, ny, nz, band, nullptr, nullptr, &g));
    size_t n = (size_t)nx * ny * nz;
    float *dd = nullptr;
    int32_t *dt = nullptr;
    int s = dev_alloc(&m->alloc, (void **)&dd, n * sizeof(float), st);
    if (s == SDF_OK) s = dev_alloc(&m->alloc, (void **)&dt, n * sizeof(int32_t), st);
    if (s == SDF_OK) s = run_compute(m, g, dd, dt, st);
    if (s != SDF_OK && m->side) cudaStreamSynchronize(m->side);
    if (s == SDF_OK) {
        cudaError_t e = cudaMemcpyAsync(dist_out_host, dd, n * sizeof(float), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(tri_out_host, dt, n * sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); s = SDF_ECUDA; }
    }
    dev_free(&m->alloc, dd, st);
    dev_free(&m->alloc, dt, st);
    return s;
}

int sdf_compute_sparse(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz, float band, int64_t brick_cap,
                       int32_t *brick_ids, float *dist_bricks, int32_t *tri_bricks, int64_t *nbricks_out, void *stream) {
    if (nbricks_out) *nbricks_out = 0;
    if (!m || !nbricks_out || brick_cap < 0) return SDF_EINVAL;
    if (brick_cap > 0 && (!brick_ids || !dist_bricks || !tri_bricks)) return SDF_EINVAL;
    if (((uintptr_t)dist_bricks & 15) || ((uintptr_t)tri_bricks & 15)) return SDF_EINVAL;
    GridParams g;
    CKS(make_grid(origin, h, nx, ny, nz, band, nullptr, nullptr, &g));
    SparseOut sp = {brick_cap, brick_ids, dist_bricks, tri_bricks, 0};
    const int s = run_compute(m, g, nullptr, nullptr, (cudaStream_t)stream, false, &sp);
    *nbricks_out = sp.count;
    return s;
}

int sdf_compute_sparse_host(sdf_mesh *m, const float origin[3], float h, int nx, int ny, int nz, float band,
                            int64_t brick_cap, int32_t *brick_ids_host, float *dist_bricks_host, int32_t *tri_bricks_host,
                            int64_t *nbricks_out, void *stream) {
    if (nbricks_out) *nbricks_out = 0;
    if (!m || !nbricks_out || brick_cap < 0) return SDF_EINVAL;
    if (brick_cap > 0 && (!brick_ids_host || !dist_bricks_host || !tri_bricks_host)) return SDF_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    GridParams g;
    CKS(make_grid(origin, h, nx, ny, nz, band, nullptr, nullptr, &g));
    // device staging for brick_cap bricks: ids, distances, triangle ids in one block
    const size_t cap = (size_t)(brick_cap > 0 ? brick_cap : 0);
    void *blk = nullptr;
    Carver c(nullptr);
    c.take<float>(cap * BRICK_CELLS); c.take<int>(cap * BRICK_CELLS); c.take<int>(cap + 1);
    int s = dev_alloc(&m->alloc, &blk, c.off, st);
    if (s != SDF_OK) return s;
    Carver d(blk);
    float *dd = d.take<float>(cap * BRICK_CELLS);
    int *dt = d.take<int>(cap * BRICK_CELLS);
    int *di = d.take<int>(cap + 1);
    SparseOut sp = {brick_cap, di, dd, dt, 0};
    s = run_compute(m, g, nullptr, nullptr, st, false, &sp);
    *nbricks_out = sp.count;
    if (s == SDF_OK && sp.count > 0) {
        const size_t n = (size_t)sp.count;
        cudaError_t e = cudaMemcpyAsync(brick_ids_host, di, n * sizeof(int), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(dist_bricks_host, dd, n * BRICK_CELLS * sizeof(float), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(tri_bricks_host, dt, n * BRICK_CELLS * sizeof(int), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); s = SDF_ECUDA; }
    } else if (s == SDF_OK) {
        cudaStreamSynchronize(st);
    }
    dev_free(&m->alloc, blk, st);
    return s;
}

int sdf_stats(sdf_mesh *m, sdf_stats_t *o) {
    if (!m || !o) return SDF_EINVAL;
    CK(cudaStreamSynchronize(m->last_stream));
    u64 all[CTR_TOTAL];            // on the stack: calls on distinct handles may run concurrently
    CK(cudaMemcpy(all, m->d_ctr, sizeof(u64) * CTR_TOTAL, cudaMemcpyDeviceToHost));
    memcpy(m->h_ctr, all, sizeof(u64) * CTR_COUNT);
    u64 *c = m->h_ctr;
    c[CTR_POLY] = c[CTR_TESTED] = c[CTR_ACCEPTED] = c[CTR_ITEMS] = c[CTR_BAND] = c[CTR_RECHECK] = 0;
    for (int s = 0; s < CTR_SLOTS; s++) {
        const u64 *q = all + CTR_SPREAD + s * 8;
        c[CTR_POLY] += q[SP_POLY]; c[CTR_TESTED] += q[SP_TESTED];
        c[CTR_ACCEPTED] += q[SP_ACCEPTED]; c[CTR_ITEMS] += q[SP_ROWS];
        c[CTR_BAND] += q[SP_BAND]; c[CTR_RECHECK] += q[SP_RECHECK];
    }
    memset(o, 0, sizeof(*o));
    o->F = m->F; o->V = m->V; o->E = m->E;
    o->edges_convex = (int64_t)c[CTR_E_CONVEX]; o->edges_concave = (int64_t)c[CTR_E_CONCAVE];
    o->edges_flat = (int64_t)c[CTR_E_FLAT];
    o->verts_pos_only = (int64_t)c[CTR_V_POS]; o->verts_neg_only = (int64_t)c[CTR_V_NEG];
    o->verts_both = (int64_t)c[CTR_V_BOTH]; o->verts_skipped = (int64_t)c[CTR_V_SKIP];
    o->verts_hemisphere = (int64_t)c[CTR_V_HEMI];
    o->weld_collisions = 0;
    o->polyhedra = (int64_t)c[CTR_POLY]; o->work_items = (int64_t)c[CTR_ITEMS];
    o->pairs_tested = (int64_t)c[CTR_TESTED]; o->pairs_accepted = (int64_t)c[CTR_ACCEPTED];
    o->bricks_active = (int64_t)c[CTR_BRICKS];
    o->bricks_total = m->last_bricks_total;
    o->band_cells = (int64_t)c[CTR_BAND]; o->fp64_rechecks = (int64_t)c[CTR_RECHECK];
    o->cdp_fallbacks = (int64_t)c[CTR_CDP_FALLBACK];
    return SDF_OK;
}

int sdf_get_table(sdf_mesh *m, int which, void *dst, size_t bytes) {
    if (!m || !dst) return SDF_EINVAL;
    const void *src = nullptr;
    size_t need = 0;
    switch (which) {
    case SDF_TABLE_CORNER_VID: src = m->cvid; need = sizeof(int) * 3 * (size_t)m->F; break;
    case SDF_TABLE_HALFEDGE_ADJ: src = m->adj; need = sizeof(int) * 3 * (size_t)m->F; break;
    case SDF_TABLE_FACE_NORMAL: src = m->fn; need = sizeof(float) * 3 * (size_t)m->F; break;
    case SDF_TABLE_VERTEX_REC: src = m->vrec; need = sizeof(VertexRec) * (size_t)m->V; break;
    case SDF_TABLE_EDGE_REC: src = m->erec; need = sizeof(EdgeRec) * (size_t)m->Elive; break;
    case SDF_TABLE_VERTEX_MINTRI: src = m->vmint; need = sizeof(int) * (size_t)m->V; break;
    default: return SDF_EINVAL;
    }
    if (bytes != need || !src) return SDF_EINVAL;
    CK(cudaStreamSynchronize(m->last_stream));
    if (which > SDF_TABLE_FACE_NORMAL) {
        CK(cudaMemcpy(dst, src, need, cudaMemcpyDeviceToHost));
        return SDF_OK;
    }
    // per-triangle tables are stored in the internal (spatially binned) order: hand them out in
    // the caller's soup order, half-edge indices included
    const size_t F = (size_t)m->F;
    int *perm = (int *)malloc(sizeof(int) * F);
    int *tmp = (int *)malloc(need);
    if (!perm || !tmp) { free(perm); free(tmp); return SDF_ENOMEM; }
    cudaError_t e = cudaMemcpy(perm, m->perm, sizeof(int) * F, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(tmp, src, need, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { free(perm); free(tmp); g_last_cuda_error = (int)e; (void)cudaGetLastError(); return SDF_ECUDA; }
    int *out = (int *)dst;          // all three tables hold 3 four-byte words per triangle
    for (size_t i = 0; i < F; i++)
        for (int k = 0; k < 3; k++) {
            int v = tmp[3 * i + k];
            if (which == SDF_TABLE_HALFEDGE_ADJ && v >= 0) v = 3 * perm[v / 3] + v % 3;
            out[3 * (size_t)perm[i] + k] = v;
        }
    free(perm); free(tmp);
    return SDF_OK;
}

} // extern "C"
